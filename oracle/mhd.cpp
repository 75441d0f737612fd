// mhd.cpp -- SURVEY.md 8(f) NEXT-4: the MHD substeps of Fig. 2 (cells 8, 10, 11; sections 3.6.1-3.7): method of
// characteristics + constrained transport (MOCCT) on Cartesian, cylindrical and spherical meshes and the shearing sheet.
//   cell 2   ghost fill of the face-centred field B (kinds of G22; the normal component keeps its boundary face)
//   cell 6   fast magnetosonic speed C_w^2 = C_s^2 + v_A^2 and the resistive limit in Eq. 59 (items 1 and 5)
//   cell 7a  gradient of the zone-centred magnetic pressure of the transverse components
//   cell 8a  star values at the zone edges by the method of characteristics (Eqs. 80-83)
//   cell 8b  electromotive forces (Eq. 84)          cell 8c  resistive term (Eq. 74)
//   cell 8d  magnetic tension on the velocities (Eq. 86) with the "Lagrangian" star values (note 14)
//   cell 10  constrained transport (Eq. 76; signs fixed by Eq. 101 P:668 and by Faraday's law: reading G35)
//   cell 11  orbital advection of B by the upstream-averaged EMF (section 3.7, Eqs. 92-107), Cartesian meshes
//            and the shearing sheet; the substeps of cell 8 then see the residual velocity v_X - v0 (reading G37)
// Curvilinear meshes (reading G38): every length is the physical one at the place where it is used -- R_x = 1 | r | r sin(theta)
// and R_z = 1 | 1 | r taken at the zone centre or at the lower Y / Z face according to where the interpolated quantity
// lives --, Eq. 76 is applied with the edge lengths and the face areas of Tab. 5, and cell 7a gets the geometric terms of
// Eqs. 87-91.  On a Cartesian mesh every R is 1.0 and the arithmetic is bit for bit what it was.
// CPU oracle, TEST INFRASTRUCTURE (see fargo_oracle.h): plain loops, one formula per line, the paper's notation.
// Directions are numbered 0, 1, 2 = X, Y, Z; (d1, d2, d3) is always a cyclic permutation, eps_d3 = v_d1 B_d2 - v_d2 B_d1.
// A field component along d lives on the LOWER d face of its cell; eps_d3 of cell q lives on the edge along d3
// at the lower-d1, lower-d2 corner of the cell, (q_d1 - 1/2, q_d2 - 1/2).
#include "oracle_impl.hpp"

namespace {

inline bool has(const oracle_ctx& c, int d) { return d == 0 ? c.hasx : d == 1 ? c.hasy : c.hasz; }
inline int ext(const oracle_ctx& c, int d) { return d == 0 ? c.TX : d == 1 ? c.TY : c.TZ; }
struct Q { int n[3]; };   // a cell: (i, j, k)
// the cell s steps along d; an absent direction has one cell, which is its own neighbour (nothing varies along it)
inline Q mv(const oracle_ctx& c, Q q, int d, int s) {
  if (!has(c, d)) return q;
  q.n[d] = (d == 0 && c.xwrap) ? c.xw(q.n[d] + s) : q.n[d] + s;
  return q;
}
inline size_t at(const oracle_ctx& c, const Q& q) { return c.id(q.n[0], q.n[1], q.n[2]); }
// R_x = 1 | r | r sin(theta) and R_z = 1 | 1 | r (Tab. 1) where a quantity that lives on the lower f face of cell q sits
// (f = 1: at the lower Y edge; f = 2: at the lower Z edge; else at the zone centre), and their reciprocals
inline double RxJ(const oracle_ctx& c, const Q& q, int f) { return c.geometry == ORC_CARTESIAN ? 1.0 : (f == 1 ? c.ye[q.n[1]] : c.yc[q.n[1]]); }
inline double RxK(const oracle_ctx& c, const Q& q, int f) { return c.geometry == ORC_SPHERICAL ? (f == 2 ? c.sin_ze[q.n[2]] : c.sin_zc[q.n[2]]) : 1.0; }
inline double RzJ(const oracle_ctx& c, const Q& q, int f) { return c.geometry == ORC_SPHERICAL ? (f == 1 ? c.ye[q.n[1]] : c.yc[q.n[1]]) : 1.0; }
inline double iRxJ(const oracle_ctx& c, const Q& q, int f) { return c.geometry == ORC_CARTESIAN ? 1.0 : (f == 1 ? c.inv_ye[q.n[1]] : c.inv_yc[q.n[1]]); }
inline double iRxK(const oracle_ctx& c, const Q& q, int f) { return c.geometry == ORC_SPHERICAL ? (f == 2 ? c.inv_sin_ze[q.n[2]] : c.invRxk[q.n[2]]) : 1.0; }
inline double iRzJ(const oracle_ctx& c, const Q& q, int f) { return c.geometry == ORC_SPHERICAL ? (f == 1 ? c.inv_ye[q.n[1]] : c.inv_yc[q.n[1]]) : 1.0; }
// physical width of cell q along d, and 1 / (distance of its centre from the centre of the zone below), for a quantity
// on the lower f face (f != d; f = d or f < 0: a zone-centred position in the two other directions)
inline double width(const oracle_ctx& c, int d, const Q& q, int f) {
  return d == 0 ? (c.dx * RxJ(c, q, f)) * RxK(c, q, f) : d == 1 ? c.LY[q.n[1]] : c.dz[q.n[2]] * RzJ(c, q, f);
}
inline double invdist(const oracle_ctx& c, int d, const Q& q, int f) {
  return d == 0 ? ((1.0 / c.dx) * iRxJ(c, q, f)) * iRxK(c, q, f) : d == 1 ? c.invDY[q.n[1]] : c.invdzc[q.n[2]] * iRzJ(c, q, f);
}
// can cell index n along d reach s_lo cells down and s_hi cells up?
inline bool fits(const oracle_ctx& c, int d, int n, int s_lo, int s_hi) {
  if (!has(c, d) || (d == 0 && c.xwrap)) return true;
  return n - s_lo >= 0 && n + s_hi < ext(c, d);
}

// van Leer slope of f along d at cell q (readings G4, G5)
inline double slope(const oracle_ctx& c, const vec& f, const Q& q, int d, int fc) {
  const Q qp = mv(c, q, d, +1);
  const double f0 = f[at(c, q)], fm = f[at(c, mv(c, q, d, -1))], fp = f[at(c, qp)];
  const double dm = (f0 - fm) * invdist(c, d, q, fc);
  const double dp = (fp - f0) * invdist(c, d, d == 0 ? q : qp, fc);   // X is uniform
  return (dm * dp <= 0.0) ? 0.0 : (2.0 * (dm * dp)) / (dm + dp);
}
// f at the lower d face of cell q at half time step, carried at speed w: Eq. 48 -- the upwind cell's value plus
// its slope times the distance to the foot of the characteristic (readings G2, G3, G6)
// (fc: the direction of the faces f lives on, which fixes the lengths on a curvilinear mesh)
inline double star(const oracle_ctx& c, const vec& f, const Q& q, int d, double w, int fc) {
  if (!has(c, d)) return f[at(c, q)];
  const Q qm = mv(c, q, d, -1);
  if (w >= 0.0) return std::fma(slope(c, f, qm, d, fc), std::fma(-w, c.dt, width(c, d, qm, fc)) * 0.5, f[at(c, qm)]);
  return std::fma(-slope(c, f, q, d, fc), std::fma(w, c.dt, width(c, d, q, fc)) * 0.5, f[at(c, q)]);
}

inline vec& V(oracle_ctx& c, int d) { return d == 0 ? (c.p.fargo_on ? c.vxres : c.vx) : d == 1 ? c.vy : c.vz; }   // G37
inline vec& B(oracle_ctx& c, int d) { return d == 0 ? c.bx : d == 1 ? c.by : c.bz; }
inline vec& EMF(oracle_ctx& c, int d) { return d == 0 ? c.emfx : d == 1 ? c.emfy : c.emfz; }

}  // namespace

// ---- cell 2: ghost fill of B.  Tangential components: as a zone-centred field in that direction.  Normal component:
// the boundary face itself is a degree of freedom of the last active cell (CT evolves it) and is left alone, except on a
// periodic axis where it IS the first active face; the ghosts beyond it are copies (outflow) or mirror images (reflecting).
static void fill_b_dir(oracle_ctx& c, vec& a, int dir, bool normal) {
  const int N = dir == 0 ? c.nx : dir == 1 ? c.ny : c.nz;
  const int ng = dir == 0 ? c.ngx : dir == 1 ? c.ngy : c.ngz;
  if (ng == 0) return;
  const int m0 = ng, m1 = ng + N;
  const int P = dir == 0 ? c.TY : c.TX, Qn = dir == 2 ? c.TY : c.TZ;
  for (int q = 0; q < Qn; ++q)
    for (int p = 0; p < P; ++p) {
      auto A = [&](int m) -> double& { return dir == 0 ? a[c.id(m, p, q)] : dir == 1 ? a[c.id(p, m, q)] : a[c.id(p, q, m)]; };
      const int lo = c.bc[dir][0], hi = c.bc[dir][1];
      for (int g = 0; g < ng; ++g) {
        if (lo == ORC_PERIODIC) A(m0 - 1 - g) = A(m1 - 1 - g);
        else if (lo == ORC_OUTFLOW) A(m0 - 1 - g) = A(m0);
        else A(m0 - 1 - g) = normal ? A(m0 + 1 + g) : A(m0 + g);          // mirror about the wall face / the wall
        if (hi == ORC_PERIODIC) A(m1 + g) = A(m0 + g);
        else if (normal) { if (g >= 1) A(m1 + g) = hi == ORC_OUTFLOW ? A(m1) : A(m1 - g); }
        else A(m1 + g) = hi == ORC_OUTFLOW ? A(m1 - 1) : A(m1 - 1 - g);
      }
    }
}
void orc_mhd_bc_fill(oracle_ctx& c) {
  for (int dir = 0; dir < 3; ++dir) {   // X, then Y, then Z: edges and corners
    fill_b_dir(c, c.bx, dir, dir == 0);
    fill_b_dir(c, c.by, dir, dir == 1);
    fill_b_dir(c, c.bz, dir, dir == 2);
  }
}

// ---- cell 6: v_A^2 = B^2 / (mu0 rho) with B at the zone centre (two-point averages of the face values) -----------------
double orc_mhd_alfven2(const oracle_ctx& c, int i, int j, int k) {
  const Q q = {{i, j, k}};
  double b2 = 0.0;
  for (int d = 0; d < 3; ++d) {
    const vec& b = d == 0 ? c.bx : d == 1 ? c.by : c.bz;
    const double bc = 0.5 * (b[at(c, q)] + b[at(c, mv(c, q, d, +1))]);
    b2 = std::fma(bc, bc, b2);
  }
  return b2 / (c.mu0 * c.rho[at(c, q)]);
}

// ---- cell 7a, MHD part: -(1/rho) d/dX_d [(B_a^2 + B_b^2) / (2 mu0)], a and b the two transverse components
// at the zone centre; the density on the face is the arithmetic mean (Eq. 53).  Applied to the result of orc_source_a.
void orc_mhd_source_a(oracle_ctx& c) {
  if (c.mhd_passive) return;
  const double dt = c.dt;
  auto pm = [&](const Q& q, int d) {   // magnetic pressure of the components transverse to d, zone centre
    double s = 0.0;
    for (int t = 1; t <= 2; ++t) {
      const int a = (d + t) % 3;
      const double bc = 0.5 * (B(c, a)[at(c, q)] + B(c, a)[at(c, mv(c, q, a, +1))]);
      s = std::fma(bc, bc, s);
    }
    return s / (2.0 * c.mu0);
  };
  for (int d = 0; d < 3; ++d) {
    if (!has(c, d)) continue;
    vec& vb = d == 0 ? c.vxb : d == 1 ? c.vyb : c.vzb;
    for (int k = 0; k < c.TZ; ++k)
      for (int j = 0; j < c.TY; ++j)
        for (int i = 0; i < c.TX; ++i) {
          const Q q = {{i, j, k}};
          if (!fits(c, d, q.n[d], 1, 0) || !fits(c, (d + 1) % 3, q.n[(d + 1) % 3], 0, 1) || !fits(c, (d + 2) % 3, q.n[(d + 2) % 3], 0, 1)) continue;
          const Q qm = mv(c, q, d, -1);
          const double il = d == 0 ? c.invLX(j, k) : d == 1 ? c.invDY[j] : c.invDZ(j, k);   // as the pressure gradient of 7a
          const double wf = (2.0 * il) / (c.rho[at(c, q)] + c.rho[at(c, qm)]);
          vb[at(c, q)] = std::fma(-dt, wf * (pm(q, d) - pm(qm, d)), vb[at(c, q)]);
        }
  }
}

// ---- cell 7a, geometric terms of B.grad B on curvilinear meshes (Eqs. 87-91), applied to v_b like the others.
// Each component of B is brought to the face of the velocity by the mean of the (two or four) face values next to it; the
// density on the face is the arithmetic mean; r, cot(theta) are those of the face.
void orc_mhd_source_curv(oracle_ctx& c) {
  if (c.mhd_passive || c.geometry == ORC_CARTESIAN) return;
  const bool sph = c.geometry == ORC_SPHERICAL;
  const double dt = c.dt, imu = 1.0 / c.mu0;
  auto avg4 = [&](const vec& b, const Q& q, int da, int db) {   // mean over q, q+e_da, q-e_db, q+e_da-e_db
    const Q qm = mv(c, q, db, -1);
    return 0.25 * (((b[at(c, q)] + b[at(c, mv(c, q, da, +1))]) + b[at(c, qm)]) + b[at(c, mv(c, qm, da, +1))]);
  };
  vec vxb = c.vxb, vyb = c.vyb, vzb = c.vzb;
  for (int k = 0; k < c.TZ; ++k)
    for (int j = 0; j < c.TY; ++j)
      for (int i = 0; i < c.TX; ++i) {
        const Q q = {{i, j, k}};
        const size_t l = at(c, q);
        const bool zok = !(sph && c.hasz) || fits(c, 2, k, 1, 1);
        if (c.hasx && fits(c, 0, i, 1, 0) && fits(c, 1, j, 0, 1) && zok) {   // v_phi on the face (i-1/2, j, k): Eqs. 87, 89
          const double wf = (2.0 * imu) / (c.rho[l] + c.rho[at(c, mv(c, q, 0, -1))]);
          const double bphi = c.bx[l], br = avg4(c.by, q, 1, 0);
          double g = br * bphi;
          if (sph && c.hasz) g = std::fma(avg4(c.bz, q, 2, 0) * bphi, c.cot_zc[k], g);
          vxb[l] = std::fma(dt, (wf * g) * c.inv_yc[j], c.vxb[l]);
        }
        if (c.hasy && fits(c, 1, j, 1, 0) && fits(c, 0, i, 0, 1) && zok) {    // v_r on the face (i, j-1/2, k): Eqs. 88, 90
          const double wf = (2.0 * imu) / (c.rho[l] + c.rho[at(c, mv(c, q, 1, -1))]);
          const double bphi = avg4(c.bx, q, 0, 1);
          double g = bphi * bphi;
          if (sph && c.hasz) { const double bth = avg4(c.bz, q, 2, 1); g = std::fma(bth, bth, g); }
          vyb[l] = std::fma(-dt, (wf * g) * c.inv_ye[j], c.vyb[l]);
        }
        if (sph && c.hasz && fits(c, 2, k, 1, 0) && fits(c, 0, i, 0, 1) && fits(c, 1, j, 0, 1)) {   // v_theta: Eq. 91
          const double wf = (2.0 * imu) / (c.rho[l] + c.rho[at(c, mv(c, q, 2, -1))]);
          const double bth = c.bz[l], br = avg4(c.by, q, 1, 2), bphi = avg4(c.bx, q, 0, 2);
          const double g = std::fma(-(bphi * bphi), c.cot_ze[k], br * bth);
          vzb[l] = std::fma(dt, (wf * g) * c.inv_yc[j], c.vzb[l]);
        }
      }
  c.vxb = vxb; c.vyb = vyb; c.vzb = vzb;
}

// ---- cells 8a-8c: star values and electromotive forces on every edge whose stencil fits ------------------------------------
// Also the "Lagrangian" star values of cell 8d (characteristic speeds -+B/sqrt(mu0 rho) only, note 14 P:1247), which live on
// the same edges: bstar[d3][0] = B_d1* from the 1.5-D problem along d2, bstar[d3][1] = B_d2* from the one along d1.
void orc_mhd_emf(oracle_ctx& c) {
  const double mu0 = c.mu0, eta = c.eta;
  if (c.p.fargo_on) {   // with orbital advection the MHD substeps see the residual velocity (reading G37)
    c.vxres = c.vx;
    for (int k = 0; k < c.TZ; ++k)
      for (int j = 0; j < c.TY; ++j)
        for (int i = 0; i < c.TX; ++i) c.vxres[c.id(i, j, k)] = c.vx[c.id(i, j, k)] - c.v0[c.rid(j, k)];
  }
  for (int d3 = 0; d3 < 3; ++d3) {
    const int d1 = (d3 + 1) % 3, d2 = (d3 + 2) % 3;
    vec &V1 = V(c, d1), &V2 = V(c, d2), &B1 = B(c, d1), &B2 = B(c, d2), &E = EMF(c, d3);
    vec &S1 = c.bstar[d3][0], &S2 = c.bstar[d3][1];
#pragma omp parallel for collapse(2) schedule(static)   // OpenMP build only: edge-independent body
    for (int k = 0; k < c.TZ; ++k)
      for (int j = 0; j < c.TY; ++j)
        for (int i = 0; i < c.TX; ++i) {
          const Q q = {{i, j, k}};
          const size_t l = at(c, q);
          E[l] = 0.0; S1[l] = B1[l]; S2[l] = B2[l];
          if (!fits(c, d1, q.n[d1], 2, 1) || !fits(c, d2, q.n[d2], 2, 1)) continue;
          const Q q1 = mv(c, q, d1, -1), q2 = mv(c, q, d2, -1), q12 = mv(c, q1, d2, -1);
          // density at the edge: the four zones around it
          const double rho = 0.25 * (((c.rho[l] + c.rho[at(c, q1)]) + c.rho[at(c, q2)]) + c.rho[at(c, q12)]);
          const double sr = std::sqrt(mu0 * rho);
          // upwind estimates of the transverse fields (superscript u): v_d1, B_d1 brought along d2 by the mean
          // v_d2 of the two faces next to the edge, and vice versa
          const double v2bar = 0.5 * (V2[l] + V2[at(c, q1)]);
          const double v1bar = 0.5 * (V1[l] + V1[at(c, q2)]);
          const double v1u = star(c, V1, q, d2, v2bar, d1), B1u = star(c, B1, q, d2, v2bar, d1);
          const double v2u = star(c, V2, q, d1, v1bar, d2), B2u = star(c, B2, q, d1, v1bar, d2);
          // (v_d2*, B_d2*): 1.5-D problem along d1, C+- = v_d1 -+ B_d1 / sqrt(mu0 rho) (Eq. 81), psi+- = v_d2 +- B_d2 / sqrt(mu0 rho)
          double v2s, B2s, v1s, B1s;
          {
            const double Cp = v1u - B1u / sr, Cm = v1u + B1u / sr;
            const double vp = star(c, V2, q, d1, Cp, d2), Bp = star(c, B2, q, d1, Cp, d2);
            const double vm = star(c, V2, q, d1, Cm, d2), Bm = star(c, B2, q, d1, Cm, d2);
            v2s = 0.5 * ((vp + vm) + (Bp - Bm) / sr);     // Eq. 83
            B2s = 0.5 * ((Bp + Bm) + sr * (vp - vm));
          }
          {   // (v_d1*, B_d1*): 1.5-D problem along d2
            const double Cp = v2u - B2u / sr, Cm = v2u + B2u / sr;
            const double vp = star(c, V1, q, d2, Cp, d1), Bp = star(c, B1, q, d2, Cp, d1);
            const double vm = star(c, V1, q, d2, Cm, d1), Bm = star(c, B1, q, d2, Cm, d1);
            v1s = 0.5 * ((vp + vm) + (Bp - Bm) / sr);
            B1s = 0.5 * ((Bp + Bm) + sr * (vp - vm));
          }
          // Eq. 84: each star value with the upwind estimate it is consistent with
          double emf = 0.5 * (((v1s * B2u + B2s * v1u) - v2s * B1u) - B1s * v2u);
          // cell 8c: - eta (curl B)_d3, plain differences
          if (eta != 0.0) {
            double J = 0.0;   // (curl B)_d3 = d(B_d2)/d(X_d1) - d(B_d1)/d(X_d2) at the edge
            if (has(c, d1)) J = (B2[l] - B2[at(c, q1)]) * invdist(c, d1, q, d2);
            if (has(c, d2)) J = J - (B1[l] - B1[at(c, q2)]) * invdist(c, d2, q, d1);
            emf = std::fma(-eta, J, emf);
          }
          E[l] = emf;
          // cell 8d, star values for the tension: the fluid and its field drift together, only -+B/sqrt(mu0 rho) is left
          // of the characteristic speed; B along the characteristic = mean of the two faces next to the edge
          {
            const double a = (0.5 * (B2[l] + B2[at(c, q1)])) / sr;      // B_d2 / sqrt(mu0 rho) at the edge
            const double vp = star(c, V1, q, d2, -a, d1), Bp = star(c, B1, q, d2, -a, d1);
            const double vm = star(c, V1, q, d2, a, d1), Bm = star(c, B1, q, d2, a, d1);
            S1[l] = 0.5 * ((Bp + Bm) + sr * (vp - vm));
          }
          {
            const double a = (0.5 * (B1[l] + B1[at(c, q2)])) / sr;
            const double vp = star(c, V2, q, d1, -a, d2), Bp = star(c, B2, q, d1, -a, d2);
            const double vm = star(c, V2, q, d1, a, d2), Bm = star(c, B2, q, d1, a, d2);
            S2[l] = 0.5 * ((Bp + Bm) + sr * (vp - vm));
          }
        }
  }
}

// ---- cell 8d: magnetic tension, Eq. 86: for v_d on the lower d face of the cell, with (d, da, db) cyclic,
//   dv_d/dt = 1/mu0 * 2/(rho + rho_-) * [ Bbar_da (B_d*(+da) - B_d*(-da)) / Delta_da + Bbar_db (B_d*(+db) - B_d*(-db)) / Delta_db ]
// B_d* on the edges along db around the face come from the 1.5-D problems along da and vice versa; the bar values are the
// four-point averages at the face centre.
void orc_mhd_lorentz(oracle_ctx& c) {
  if (c.mhd_passive) return;
  const double dt = c.dt;
  for (int d = 0; d < 3; ++d) {
    if (!has(c, d)) continue;
    const int da = (d + 1) % 3, db = (d + 2) % 3;
    vec& v = d == 0 ? c.vx : d == 1 ? c.vy : c.vz;
    const vec &Ba = B(c, da), &Bb = B(c, db);
    const vec &Sa = c.bstar[db][0];   // B_d* on the edges along db (d3 = db: d1 = d, d2 = da)
    const vec &Sb = c.bstar[da][1];   // B_d* on the edges along da (d3 = da: d1 = db, d2 = d)
    vec out = v;
    for (int k = 0; k < c.TZ; ++k)
      for (int j = 0; j < c.TY; ++j)
        for (int i = 0; i < c.TX; ++i) {
          const Q q = {{i, j, k}};
          if (!fits(c, d, q.n[d], 2, 1) || !fits(c, da, q.n[da], 2, 2) || !fits(c, db, q.n[db], 2, 2)) continue;
          const size_t l = at(c, q);
          const Q qm = mv(c, q, d, -1), qa = mv(c, q, da, +1), qb = mv(c, q, db, +1);
          const double Bbar_a = 0.25 * (((Ba[l] + Ba[at(c, qa)]) + Ba[at(c, qm)]) + Ba[at(c, mv(c, qm, da, +1))]);
          const double Bbar_b = 0.25 * (((Bb[l] + Bb[at(c, qb)]) + Bb[at(c, qm)]) + Bb[at(c, mv(c, qm, db, +1))]);
          double acc = 0.0;
          if (has(c, da)) acc = Bbar_a * ((Sa[at(c, qa)] - Sa[l]) / width(c, da, q, d));
          if (has(c, db)) acc = std::fma(Bbar_b, (Sb[at(c, qb)] - Sb[l]) / width(c, db, q, d), acc);
          const double wf = 2.0 / (c.mu0 * (c.rho[l] + c.rho[at(c, qm)]));
          out[l] = std::fma(dt, wf * acc, v[l]);
        }
    v = out;
  }
}

// ---- cell 10: constrained transport.  d(B_d)/dt = (curl eps)_d on the lower d face of the cell:
//   (eps_db(+da) - eps_db) / Delta_da - (eps_da(+db) - eps_da) / Delta_db        (Eq. 76 with the signs of Eq. 101; G35)
// Every edge value enters two faces of a cell with opposite signs: div B keeps its value to rounding.
void orc_mhd_ct(oracle_ctx& c) {
  const double dt = c.dt;
  if (c.geometry != ORC_CARTESIAN) {
    // Eq. 76 proper: d(B S)/dt = circulation of eps around the face, with the physical edge lengths and Tab. 5's areas.
    //   Z edge at (i-1/2, j-1/2, k): lZ = dz R_z(edge j);  X edge at (i, j-1/2, k-1/2): lX = dx R_x(edge j, edge k);  Y edge: LY[j]
    auto lZ = [&](int j, int k) { return c.dz[k] * (c.geometry == ORC_SPHERICAL ? c.ye[j] : 1.0); };
    auto lX = [&](int j, int k) { return (c.dx * c.ye[j]) * (c.geometry == ORC_SPHERICAL ? c.sin_ze[k] : 1.0); };
    vec bx = c.bx, by = c.by, bz = c.bz;
    for (int k = 0; k < c.TZ; ++k)
      for (int j = 0; j < c.TY; ++j)
        for (int i = 0; i < c.TX; ++i) {
          const Q q = {{i, j, k}};
          const size_t l = at(c, q);
          const size_t li = at(c, mv(c, q, 0, +1)), lj = at(c, mv(c, q, 1, +1)), lk = at(c, mv(c, q, 2, +1));
          if (fits(c, 0, i, 2, 1) && fits(c, 1, j, 2, 2) && fits(c, 2, k, 2, 2)) {
            double circ = 0.0;
            if (c.hasy) circ = c.emfz[lj] * lZ(j + 1, k) - c.emfz[l] * lZ(j, k);
            if (c.hasz) circ = circ - (c.emfy[lk] - c.emfy[l]) * c.LY[j];
            bx[l] = std::fma(dt, circ / c.Sx(j, k), c.bx[l]);
          }
          if (fits(c, 1, j, 2, 1) && fits(c, 2, k, 2, 2) && fits(c, 0, i, 2, 2)) {
            double circ = 0.0;
            if (c.hasz) circ = c.emfx[lk] * lX(j, k + 1) - c.emfx[l] * lX(j, k);
            if (c.hasx) circ = circ - (c.emfz[li] - c.emfz[l]) * lZ(j, k);
            by[l] = std::fma(dt, circ / c.Sy(j, k), c.by[l]);
          }
          if (fits(c, 2, k, 2, 1) && fits(c, 0, i, 2, 2) && fits(c, 1, j, 2, 2)) {
            double circ = 0.0;
            if (c.hasx) circ = (c.emfy[li] - c.emfy[l]) * c.LY[j];
            if (c.hasy) circ = circ - (c.emfx[lj] * lX(j + 1, k) - c.emfx[l] * lX(j, k));
            bz[l] = std::fma(dt, circ / c.Sz(j, k), c.bz[l]);
          }
        }
    c.bx = bx; c.by = by; c.bz = bz;
    return;
  }
  for (int d = 0; d < 3; ++d) {
    const int da = (d + 1) % 3, db = (d + 2) % 3;
    vec& b = B(c, d);
    const vec &Eb = EMF(c, db), &Ea = EMF(c, da);
    for (int k = 0; k < c.TZ; ++k)
      for (int j = 0; j < c.TY; ++j)
        for (int i = 0; i < c.TX; ++i) {
          const Q q = {{i, j, k}};
          if (!fits(c, d, q.n[d], 2, 1) || !fits(c, da, q.n[da], 2, 2) || !fits(c, db, q.n[db], 2, 2)) continue;
          const size_t l = at(c, q);
          double curl = 0.0;
          if (has(c, da)) curl = (Eb[at(c, mv(c, q, da, +1))] - Eb[l]) / width(c, da, q, d);
          if (has(c, db)) curl = curl - (Ea[at(c, mv(c, q, db, +1))] - Ea[l]) / width(c, db, q, d);
          b[l] = std::fma(dt, curl, b[l]);
        }
  }
}

// div B of a cell (Eq. 75 summed over its six faces, divided by the volume): the CT invariant
double orc_mhd_divb(const oracle_ctx& c, int i, int j, int k) {
  const Q q = {{i, j, k}};
  if (c.geometry != ORC_CARTESIAN) {   // (sum of B S over the six faces) / V with Tab. 5's areas and volume
    double s = 0.0;
    if (c.hasx) s += (c.bx[at(c, mv(c, q, 0, +1))] - c.bx[at(c, q)]) * c.Sx(j, k);
    if (c.hasy) s += c.by[at(c, mv(c, q, 1, +1))] * c.Sy(j + 1, k) - c.by[at(c, q)] * c.Sy(j, k);
    if (c.hasz) s += c.bz[at(c, mv(c, q, 2, +1))] * c.Sz(j, k + 1) - c.bz[at(c, q)] * c.Sz(j, k);
    return s * c.invV(j, k);
  }
  double s = 0.0;
  for (int d = 0; d < 3; ++d) {
    if (!has(c, d)) continue;
    const vec& b = d == 0 ? c.bx : d == 1 ? c.by : c.bz;
    s += (b[at(c, mv(c, q, d, +1))] - b[at(c, q)]) / width(c, d, q, d);
  }
  return s;
}

// ---- cell 11: orbital advection of B (section 3.7).  d/dt B = curl (v0 x B) with v0 = v0(Y, Z) along X, integrated
// over the whole step with the upstream average of the EMF (Eq. 96): the time integral of eps_Z at the edge
// (i-1/2, j-1/2, k) is DX times the integral of B_Y over the arc of s = v0 dt / DX cells upstream of it, i.e. over
// "as many zones as necessary" -- N = nint(s) whole zones, summed one after the other -- plus the residual
// xi = s - N of a zone from the parabolic reconstruction of the orbital advection; v0 on a face is
// the mean of the two zones next to it.  eps_Y = -v0 B_Z likewise on the edges (i-1/2, j, k-1/2); eps_X = 0.
// The constrained-transport update with these integrals shifts B_Y and B_Z like zone-centred quantities (Eq. 103) and
// gives B_X the shift plus the shear term (Eqs. 94, 104-107); div B keeps its value to rounding.
// phi[i] of a row g = (integral of g over the arc upstream of the face i-1/2) / DX.
static void arc_integrals(int n, const double* g, double s, double* phi) {
  if (!std::isfinite(s) || std::fabs(s) > 4.0 * n) { for (int i = 0; i < n; ++i) phi[i] = s; return; }   // a blown-up run: no loop over ~inf zones
  const double N = std::floor(s + 0.5), xi = s - N;   // reading G11
  const int Ni = (int)N;
  std::vector<double> gs(n);
  oracle_ppa_star(n, g, xi, gs.data());                // gs[c]: mean of g over the part of the upwind zone that crosses face c+1/2
  auto w = [n](int i) { int m = i % n; return m < 0 ? m + n : m; };
  for (int i = 0; i < n; ++i) {                        // face i-1/2 = face (i-1)+1/2
    double S = 0.0;
    if (Ni > 0) for (int m = 0; m < Ni; ++m) S = S + g[w(i - 1 - m)];
    if (Ni < 0) for (int m = 1; m <= -Ni; ++m) S = S - g[w(i - 1 + m)];
    phi[i] = std::fma(xi, gs[w(i - 1 - Ni)], S);
  }
}
void orc_mhd_orbital(oracle_ctx& c) {
  if (!c.p.fargo_on) return;
  const int n = c.TX;   // orbital advection needs a wrapped X axis: TX = nx
  const double dt = c.dt;
  const bool cart = c.geometry == ORC_CARTESIAN;
  vec &PZ = c.emfz, &PY = c.emfy;   // reused: the arc integrals on the Z edges (of B_Y) and on the Y edges (of B_Z)
  std::vector<double> g(n), phi(n);
  for (int k = 0; k < c.TZ; ++k)
    for (int j = 0; j < c.TY; ++j) {
      const size_t base = c.id(0, j, k);
      for (int i = 0; i < n; ++i) { PZ[base + i] = 0.0; PY[base + i] = 0.0; }
      if (!c.hasy || j >= 1) {   // Z edges of the Y face j-1/2: v0 = mean of the rings j-1 and j
        const double v0f = c.hasy ? 0.5 * (c.v0[c.rid(j, k)] + c.v0[c.rid(j - 1, k)]) : c.v0[c.rid(j, k)];
        for (int i = 0; i < n; ++i) g[i] = c.by[base + i];
        arc_integrals(n, g.data(), (v0f * dt) * invdist(c, 0, Q{{0, j, k}}, 1), phi.data());   // zones of the Y face's own arc length
        for (int i = 0; i < n; ++i) PZ[base + i] = phi[i];
      }
      if (!c.hasz || k >= 1) {   // Y edges of the Z face k-1/2
        const double v0f = c.hasz ? 0.5 * (c.v0[c.rid(j, k)] + c.v0[c.rid(j, k - 1)]) : c.v0[c.rid(j, k)];
        for (int i = 0; i < n; ++i) g[i] = c.bz[base + i];
        arc_integrals(n, g.data(), (v0f * dt) * invdist(c, 0, Q{{0, j, k}}, 2), phi.data());
        for (int i = 0; i < n; ++i) PY[base + i] = phi[i];
      }
    }
  for (int k = 0; k < c.TZ; ++k)
    for (int j = 0; j < c.TY; ++j) {
      if ((c.hasy && (j < 1 || j + 1 >= c.TY)) || (c.hasz && (k < 1 || k + 1 >= c.TZ))) continue;
      const size_t base = c.id(0, j, k);
      for (int i = 0; i < n; ++i) {
        const int ip = c.xw(i + 1);
        const size_t l = base + i, lp = base + ip;
        // B_X: DX [ (PZ(j+1) - PZ(j)) / DY + (PY(k+1) - PY(k)) / DZ ]   (Eq. 104 and its Z counterpart)
        double d = 0.0;
        if (cart) {
          if (c.hasy) d = (c.dx * (PZ[c.id(i, j + 1, k)] - PZ[l])) / c.LY[j];
          if (c.hasz) d = d + (c.dx * (PY[c.id(i, j, k + 1)] - PY[l])) / c.dz[k];
        } else {   // cylindrical: the same circulation with each edge's own arc length (Eq. 105), over the area of the face
          const Q q = {{i, j, k}}, qj = {{i, j + 1, k}}, qk = {{i, j, k + 1}};
          if (c.hasy) d = (width(c, 0, qj, 1) * PZ[c.id(i, j + 1, k)]) * c.dz[k] - (width(c, 0, q, 1) * PZ[l]) * c.dz[k];
          if (c.hasz) d = d + (width(c, 0, qk, 2) * PY[c.id(i, j, k + 1)] - width(c, 0, q, 2) * PY[l]) * c.LY[j];
          d = d / c.Sx(j, k);
        }
        c.bx[l] = c.bx[l] + d;
        c.by[l] = c.by[l] - (PZ[lp] - PZ[l]);          // Eq. 101
        c.bz[l] = c.bz[l] - (PY[lp] - PY[l]);
      }
    }
}
