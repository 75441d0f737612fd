// kernels.h -- launchers of the CUDA kernels of one hydrodynamic update (host-callable, templated
// on the arithmetic type, instantiated for double and float in the k_*.cu files).
// Every launcher enqueues on `s` and returns the number of kernels it launched.
#pragma once
#include <string>
#include "common.cuh"

namespace fg {

enum { F_RHO = 1, F_E = 2, F_VX = 4, F_VY = 8, F_VZ = 16 };

// cells 2 / 9: ghost fill of the fields in `mask`, X then Y then Z
template <typename T> int launch_bc(const Dev<T>& d, const State<T>& st, int mask, cudaStream_t s);
// cell 3: v0_jk = (max_i vx + min_i vx)/2 (Eq. 72)
template <typename T> int launch_vmean(const Dev<T>& d, const T* vx, T* v0, cudaStream_t s);
// cell 5: potential of the star and the planet at cell centres; cphi, sphi = cos, sin of the planet's azimuth
// (ppos != nullptr: the planet's (x_p, y_p) are read from that device address instead)
template <typename T> int launch_potential(const Dev<T>& d, T* phi, T gm_star, T gm_planet, T xp, T yp, T eps2,
                                           const T* ppos, cudaStream_t s);
// live planets (NEXT-2, k_planets.cu): cell 5 with the planets where they are now (device state); cell 5a = gas force
// (block partials in `part`, planets_blocks() x 3 MAXPL doubles), kick and one Cash-Karp step over ctl->dt
int planets_blocks(int ny, int nz);
template <typename T> int launch_potential_live(const Dev<T>& d, T* phi, T gm_star, const PlanetsDev* pl, int npl, cudaStream_t s);
template <typename T> int launch_planets_update(const Dev<T>& d, const T* rho, PlanetsDev* pl, int npl, int mode, double* part,
                                                double gm_star, double omega, cudaStream_t s);
// cell 5b, Eq. 44: vx -= dom R_x(j,k) on the whole array; the live planets follow into the new frame
template <typename T> int launch_frame_change(const Dev<T>& d, T* vx, double dom, PlanetsDev* pl, int npl, cudaStream_t s);
// diagnostics: per-block partial sums of mass, Tab. 2 momenta and internal energy: part[planets_blocks()][5]
template <typename T> int launch_diagnostics(const Dev<T>& d, const State<T>& st, double* part, cudaStream_t s);
// the same with the partials in a file-scope device array and the final sums added on the device into out_device[5]
// (k_noalloc.cu: no allocation, no synchronisation); launches, or -1 (mesh beyond the array) / -2 (CUDA error) + err
template <typename T> int launch_diagnostics_noalloc(const Dev<T>& d, const State<T>& st, double* out_device, cudaStream_t s,
                                                     std::string& err);
long long diagnostics_noalloc_max_rings();
// cell 6: Eq. 59 + Eq. 73 -> ctl->dt (device resident)
enum { DT_BOTH = 0, DT_FINISH = 1, DT_CELLS = 2 };   // per-cell max + finish | finish only | per-cell max only
// MHD (NEXT-4): the face-centred field for the fast magnetosonic speed, 4 eta for the resistive limit (bx = nullptr: off)
template <typename T> struct MhdDt { const T *bx, *by, *bz; T mu0, eta4; int passive; };
template <typename T> int launch_dt(const Dev<T>& d, const State<T>& st, const T* v0, cudaStream_t s, int mode = DT_BOTH,
                                    const MhdDt<T>* mhd = nullptr);
// cell 7a: st -> vb[3]
template <typename T> int launch_source_a(const Dev<T>& d, const State<T>& st, const T* phi, T* vxb, T* vyb, T* vzb,
                                          cudaStream_t s);
// cell 7b: (rho, e, vb) -> vc[3], ec
template <typename T> int launch_source_b(const Dev<T>& d, const State<T>& st, const T* vxb, const T* vyb,
                                          const T* vzb, T* vxc, T* vyc, T* vzc, T* ec, cudaStream_t s);
// cells 7b + 7c fused (adiabatic): (rho, e, vb) -> vc[3], ed; ed may alias st.e (each thread reads only its own e)
template <typename T> int launch_source_bc(const Dev<T>& d, const State<T>& st, const T* vxb, const T* vyb,
                                           const T* vzb, T* vxc, T* vyc, T* vzc, T* ed, cudaStream_t s);
// cell 7c: (vc, ec) -> ed
template <typename T> int launch_source_c(const Dev<T>& d, const T* vxc, const T* vyc, const T* vzc, const T* ec,
                                          T* ed, cudaStream_t s);
// cells 7a-7c in ONE pass (3-D meshes, wrapped X with an even nx, no viscosity): st -> out.{e, vx, vy, vz}
template <typename T> bool source_fused_ok(const Dev<T>& d);
template <typename T> int launch_source_fused(const Dev<T>& d, const State<T>& st, const T* phi, const State<T>& out,
                                              cudaStream_t s);
// cell 7d (2-D cylindrical): (rho, vc) -> vd, with the stress tensor in tpp, trr, tpr
template <typename T> int launch_source_d(const Dev<T>& d, const T* rho, const T* vxc, const T* vyc, T* tpp, T* trr,
                                          T* tpr, T* vxd, T* vyd, cudaStream_t s);

// cell 7d on a 3-D mesh, all three geometries (Eqs. B1-B6): (rho, vc) -> vd; t[0..5] = xx yy zz xy xz yz
template <typename T> int launch_source_d3(const Dev<T>& d, const T* rho, const T* vxc, const T* vyc, const T* vzc,
                                           T* const* t, T* vxd, T* vyd, T* vzd, cudaStream_t s);

// the same in ONE pass on a wrapped X axis, active cells only (the ghost fill of cell 9 follows): (rho, vc) -> vd
template <typename T> bool source_d3_fused_ok(const Dev<T>& d);
template <typename T> int launch_source_d3_fused(const Dev<T>& d, const T* rho, const T* vxc, const T* vyc, const T* vzc,
                                                 T* vxd, T* vyd, T* vzd, cudaStream_t s);

// cells 12a-12c: one directional sweep.  first != 0: the momenta are formed from the state (12a fused).
template <typename T> struct SweepArgs {
  State<T> st;        // state: e and velocities for the momenta (first pass); the frozen face velocities
  const T* srho;      // density read by this pass (the state's on the first pass)
  T* drho;            // density written by this pass
  const T* sq[8];     // the nq transported quantities read (compacted; unused on the first pass)
  T* dq[8];           // ... and written
  const T* v0;        // ring mean velocity or nullptr
  int nq;             // transported quantities besides rho (<= 7)
  int slot[8];        // what each one is: 0 = e, 1..6 = pxm pxp pym pyp pzm pzp
  int first;
};
template <typename T> int launch_sweep(const Dev<T>& d, const SweepArgs<T>& a, int dir, cudaStream_t s);
// cell 12a alone (only when X is absent): momenta of the Y and Z directions into S.q[3..6]
template <typename T> int launch_momenta(const Dev<T>& d, const State<T>& st, const QSet<T>& S, cudaStream_t s);
// orbital advection: PPA fractional sweep (Eq. 70) with the integer shift (Eq. 69) folded into the store index
template <typename T> int launch_orbital(const Dev<T>& d, const SweepArgs<T>& a, T* nshift_out, cudaStream_t s);
// cell 12d: Eq. 51; then the clock advances
template <typename T> int launch_newvel(const Dev<T>& d, const T* rho, const QSet<T>& set, const State<T>& st,
                                        cudaStream_t s);
// cell 12d fused with cell 6 of the next update (no orbital advection, X wrapped, Y and Z periodic): Eq. 51, then the
// per-cell rate of Eq. 59 for the new state into ctl->m2bits; launch_dt(..., DT_FINISH) finishes it
template <typename T> bool newvel_dt_ok(const Dev<T>& d);
template <typename T> int launch_newvel_dt(const Dev<T>& d, const T* rho, const T* e, const QSet<T>& set, const State<T>& st,
                                           cudaStream_t s);
template <typename T> int launch_copy(const Dev<T>& d, const T* src, T* dst, cudaStream_t s);
int launch_advance(Ctl* ctl, double t_stop, cudaStream_t s);
// slabs: retake the t_stop clip flag after ctl->dt was all-reduced (min) over the slabs
int launch_dt_sync(Ctl* ctl, double t_stop, bool single, cudaStream_t s);
int launch_dt_min(Ctl* ctl, const double* other, cudaStream_t s);   // ctl->dt = min(ctl->dt, *other)
// out[n] = rdiv(a[n], b[n]): the kernels' branch-free division, exposed for its self-test
int launch_selftest_div(const double* a, const double* b, double* out, long long n, cudaStream_t s);

// MHD on 3-D Cartesian meshes (NEXT-4, k_mhd.cu): ghost fill of B; magnetic pressure in 7a (on v_b, in place); star values
// and EMFs (emf[3]; bstar[6]: [2 d3] = B_d1*, [2 d3 + 1] = B_d2* on the edges along d3); tension (8d) and CT (10), in place
template <typename T> int launch_bc_b(const Dev<T>& d, T* bx, T* by, T* bz, cudaStream_t s);
template <typename T> int launch_mhd_pressure(const Dev<T>& d, const T* rho, T* bx, T* by, T* bz, T* vxb, T* vyb, T* vzb, double mu0,
                                              cudaStream_t s);
template <typename T> int launch_mhd_emf(const Dev<T>& d, const T* rho, T* vx, T* vy, T* vz, T* bx, T* by, T* bz, T* const* emf,
                                         T* const* bstar, double mu0, double eta, cudaStream_t s);
template <typename T> int launch_mhd_tension(const Dev<T>& d, const T* rho, T* const* b, T* const* bstar, T* vx, T* vy, T* vz,
                                             double mu0, cudaStream_t s);
template <typename T> int launch_mhd_ct(const Dev<T>& d, T* const* emf, T* bx, T* by, T* bz, cudaStream_t s);
// cell 11 (section 3.7): vres = vx - v0 for cell 8; arc integrals of B_Y, B_Z (into PZ, PY) and the CT update with them
template <typename T> int launch_mhd_resid(const Dev<T>& d, const T* vx, const T* v0, T* vres, cudaStream_t s);
template <typename T> int launch_mhd_orbital(const Dev<T>& d, const T* v0, T* bx, T* by, T* bz, T* PZ, T* PY, cudaStream_t s);

// active cells <-> ghosted, padded device layout
template <typename T> int launch_scatter(const Dev<T>& d, const T* active, T* full, cudaStream_t s);
template <typename T> int launch_gather(const Dev<T>& d, const T* full, T* active, cudaStream_t s);
template <typename T> int launch_unpad(const Dev<T>& d, const T* full, T* out, cudaStream_t s);

}  // namespace fg
