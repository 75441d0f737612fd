// oracle_impl.hpp -- internal state of the CPU oracle (TEST INFRASTRUCTURE, see fargo_oracle.h).
// Plain fp64, single thread, one triple loop per box of Fig. 2.  No blocking, no fusion.
#pragma once
#include <cmath>
#include <cstring>
#include <string>
#include <vector>

#include "fargo_oracle.h"

typedef std::vector<double> vec;

struct oracle_ctx {
  // ---- mesh --------------------------------------------------------------
  int nx, ny, nz;        // active cells
  int ng;                // ghost layers requested (3)
  int ngx, ngy, ngz;     // ghost layers actually carried: 0 for an absent direction or wrapped X
  int TX, TY, TZ;        // allocated extents
  int geometry, eos;
  int bc[3][2];
  bool xwrap;            // X periodic: no ghosts, index algebra wraps
  bool hasx, hasy, hasz; // direction present (N > 1)
  double dx, xmin;
  oracle_params p;
  bool has_pot;          // star or planet potential present (cyl / sph only)
  bool shear;            // shearing sheet: `geometry` is then ORC_CARTESIAN (same metric, Tab. 5) and
                         // only Tab. 2's X momentum and Eq. 29's source term differ (reading G32)

  // 1-D tables, ghost-inclusive.  j tables have TY (+1 for edges) entries, k tables TZ (+1).
  vec ye, yc, ze, zc;                  // edges and centres (centre = mean of edges, reading G26)
  vec inv_ye, inv_yc;
  vec LY, invLY, DY, invDY;            // cell width in Y; centre distance yc[j]-yc[j-1]
  vec dz, invdz, dzc, invdzc;          // coordinate width in Z; centre distance zc[k]-zc[k-1]
  vec sxj, sxk, syj, syk, szj, szk, invVj, inv_syk;   // Tab. 5
  vec Rxj, Rxk, invRxj, invRxk;        // R_x(j,k) = Rxj[j]*Rxk[k]  (1 | r | r sin(theta))
  vec LXj, invLXj;                     // LX(j,k) = LXj[j]*Rxk[k],  LXj = dx*Rxj
  vec Rzj, invRzj;                     // R_z(j) = 1 | 1 | r
  vec sin_zc, sin_ze, cos_zc, cos_ze, cot_ze;   // host libm tables (no transcendental elsewhere)
  vec cot_zc, inv_sin_ze;                        // cos/sin at centres, 1/sin at edges (3-D viscous stress)
  vec cos_xc, sin_xc;                  // cos/sin of the azimuth of cell centres

  // ---- fields, ghost-inclusive, X fastest ----------------------------------------------------
  // ---- live planets (NEXT-2, planets.cpp) ------------------------------------------------------
  int npl = 0, force_mode = 0;
  double pl_gconst = 1.0;
  double pl_gm[ORC_MAX_PLANETS], pl_eps[ORC_MAX_PLANETS];
  double pl_x[ORC_MAX_PLANETS][3], pl_v[ORC_MAX_PLANETS][3], pl_f[ORC_MAX_PLANETS][3];
  vec Vj;                              // 1 / invVj: V(j,k) = Vj[j] * syk[k] (Tab. 5)

  // ---- MHD (NEXT-4, mhd.cpp): face-centred field, edge-centred electromotive forces and star values ----------
  bool mhd = false, mhd_passive = false;   // passive: B is advected and diffused but exerts no force
  double mu0 = 1.0, eta = 0.0;             // permeability, resistivity (Eq. 5)
  vec bx, by, bz, emfx, emfy, emfz;
  vec bstar[3][2];
  vec vxres;                               // v_X - v0: what cell 8 sees under orbital advection (reading G37)

  vec rho, e, vx, vy, vz;              // state
  vec phi;                             // potential at centres (cell 5)
  vec vxb, vyb, vzb;                   // after 7a
  vec vxc, vyc, vzc, ec;               // after 7b
  vec ed;                              // after 7c
  vec vxd, vyd, vzd;                   // after 7d (2-D cylindrical; 3-D in all three geometries)
  vec pxm, pxp, pym, pyp, pzm, pzp;    // left/right momenta (Eqs. 49-50)
  vec v0;                              // ring mean velocity, TY*TZ
  vec nshift;                          // integer shift per ring (stored as double), TY*TZ
  vec xi;                              // fractional shift per ring
  double t, dt;
  long long nsteps;
  bool midstep;

  inline size_t id(int i, int j, int k) const { return (size_t)i + (size_t)TX * ((size_t)j + (size_t)TY * (size_t)k); }
  inline size_t rid(int j, int k) const { return (size_t)j + (size_t)TY * (size_t)k; }
  // X neighbour with wrap when periodic; otherwise plain (callers stay in range)
  inline int xw(int i) const { if (!xwrap) return i; int m = i % nx; return m < 0 ? m + nx : m; }
  inline size_t ncell() const { return (size_t)TX * TY * TZ; }

  inline double LX(int j, int k) const { return LXj[j] * Rxk[k]; }
  inline double invLX(int j, int k) const { return invLXj[j] * invRxk[k]; }
  inline double LZ(int j, int k) const { return dz[k] * Rzj[j]; }
  inline double invLZ(int j, int k) const { return invdz[k] * invRzj[j]; }
  inline double invDZ(int j, int k) const { return invdzc[k] * invRzj[j]; }
  inline double Sx(int j, int k) const { return sxj[j] * sxk[k]; }
  inline double Sy(int j, int k) const { return syj[j] * syk[k]; }
  inline double Sz(int j, int k) const { return szj[j] * szk[k]; }
  inline double invV(int j, int k) const { return invVj[j] * inv_syk[k]; }
  inline double Rx(int j, int k) const { return Rxj[j] * Rxk[k]; }
  inline double invRx(int j, int k) const { return invRxj[j] * invRxk[k]; }

  // active index ranges
  inline int i0() const { return ngx; } inline int i1() const { return ngx + nx; }
  inline int j0() const { return ngy; } inline int j1() const { return ngy + ny; }
  inline int k0() const { return ngz; } inline int k1() const { return ngz + nz; }
};

// stages (one function per box of Fig. 2)
void orc_build_tables(oracle_ctx& c, const oracle_mesh& m);
void orc_bc_fill(oracle_ctx& c, vec& rho, vec& e, vec& vx, vec& vy, vec& vz);
void orc_vmean(oracle_ctx& c);
void orc_potential(oracle_ctx& c);
double orc_compute_dt(oracle_ctx& c, bool* clipped);
void orc_source_a(oracle_ctx& c);
void orc_source_b(oracle_ctx& c);
void orc_source_c(oracle_ctx& c);
void orc_source_d(oracle_ctx& c);
bool orc_visc3d_on(const oracle_ctx& c);
void orc_source_d3(oracle_ctx& c);   // viscosity3d.cpp
void orc_momenta(oracle_ctx& c);
void orc_sweep(oracle_ctx& c, int dir);
void orc_orbital_frac(oracle_ctx& c);
void orc_orbital_shift(oracle_ctx& c);
void orc_newvel(oracle_ctx& c);
void orc_planets_update(oracle_ctx& c);   // planets.cpp, cell 5a
// mhd.cpp (NEXT-4; Cartesian meshes)
void orc_mhd_bc_fill(oracle_ctx& c);
double orc_mhd_alfven2(const oracle_ctx& c, int i, int j, int k);
void orc_mhd_source_a(oracle_ctx& c);
void orc_mhd_source_curv(oracle_ctx& c);
void orc_mhd_emf(oracle_ctx& c);
void orc_mhd_lorentz(oracle_ctx& c);
void orc_mhd_ct(oracle_ctx& c);
void orc_mhd_orbital(oracle_ctx& c);
double orc_mhd_divb(const oracle_ctx& c, int i, int j, int k);
