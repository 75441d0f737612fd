// transport.cpp -- the transport step, box 12 of Fig. 2: momenta (12a, Eqs. 49-50), van Leer upwind
// star values (12b, Eq. 48), conservative updates per direction (12c, Eqs. 41-43, 45-47) with
// consistent transport, new velocities (12d, Eq. 51).
// CPU oracle, TEST INFRASTRUCTURE (see fargo_oracle.h).
#include "oracle_impl.hpp"

// ---- 1-D primitives ------------------------------------------------------------------------------
// van Leer slope (formula after Eq. 48) per unit length; zero when the one-sided
// differences have opposite signs or one of them vanishes (reading G4).  Differences are taken over
// centre-to-centre distances (reading G5): invd[m] = 1/(c_m - c_{m-1}).
extern "C" void oracle_vanleer_slopes(int n, const double* f, const double* invd, double* a) {
  for (int m = 0; m < n; ++m) a[m] = 0.0;
  for (int m = 1; m + 1 < n; ++m) {
    const double dm = (f[m] - f[m - 1]) * invd[m];
    const double dp = (f[m + 1] - f[m]) * invd[m + 1];
    a[m] = (dm * dp <= 0.0) ? 0.0 : (2.0 * (dm * dp)) / (dm + dp);
  }
}

// Upwind value at half time step on the lower face of cell m (Eq. 48; readings G2, G3, G6):
// w >= 0: the upwind cell is m-1;  w < 0: it is m, and the width is that of the upwind cell.
extern "C" void oracle_vanleer_star(int n, const double* f, const double* a, const double* len, const double* w,
                                    double dt, double* fstar) {
  fstar[0] = f[0];
  for (int m = 1; m < n; ++m)
    fstar[m] = (w[m] >= 0.0) ? std::fma(a[m - 1], std::fma(-w[m], dt, len[m - 1]) * 0.5, f[m - 1])
                             : std::fma(-a[m], std::fma(w[m], dt, len[m]) * 0.5, f[m]);
}

// ---- 12a: left / right momenta with the quantities of Tab. 2 -----------------------
void orc_momenta(oracle_ctx& c) {
  const double om = (c.geometry == ORC_CARTESIAN) ? 0.0 : c.p.omega_frame;
#pragma omp parallel for collapse(2) schedule(static)   // OpenMP build only (liboracle_omp.so): cell-independent body
  for (int k = 0; k < c.TZ; ++k)
    for (int j = 0; j < c.TY; ++j) {
      // Tab. 2: the term added to R_x v_x; shearing sheet: 2 Omega_f y at the cell centre (G32)
      const double rx = c.Rx(j, k), rx2om = c.shear ? (2.0 * c.p.omega_frame) * c.yc[j] : (rx * rx) * om, rz = c.Rzj[j];
      for (int i = 0; i < c.TX; ++i) {
        const size_t l = c.id(i, j, k);
        const double r = c.rho[l];
        const bool ipok = c.xwrap || i + 1 < c.TX;
        const double vxp = (c.hasx && ipok) ? c.vx[c.id(c.xw(i + 1), j, k)] : c.vx[l];
        const double vyp = (c.hasy && j + 1 < c.TY) ? c.vy[c.id(i, j + 1, k)] : c.vy[l];
        const double vzp = (c.hasz && k + 1 < c.TZ) ? c.vz[c.id(i, j, k + 1)] : c.vz[l];
        c.pxm[l] = r * std::fma(rx, c.vx[l], rx2om);
        c.pxp[l] = r * std::fma(rx, vxp, rx2om);
        c.pym[l] = r * c.vy[l];
        c.pyp[l] = r * vyp;
        c.pzm[l] = r * (rz * c.vz[l]);
        c.pzp[l] = r * (rz * vzp);
      }
    }
}

// ---- 12b + 12c: one directional sweep of rho and of every transported quantity --------------------
// Line by line along `dir`.  In X with wrap the line is extended by two periodic copies per side.
void orc_sweep(oracle_ctx& c, int dir) {
  const bool has = dir == 0 ? c.hasx : dir == 1 ? c.hasy : c.hasz;
  if (!has) return;
  const double dt = c.dt;
  const int T = dir == 0 ? c.TX : dir == 1 ? c.TY : c.TZ;
  const bool wrap = (dir == 0 && c.xwrap);
  const int H = wrap ? 2 : 0;          // periodic halo added to the line
  const int n = T + 2 * H;
  const int P = dir == 0 ? c.TY : c.TX, Q = dir == 2 ? c.TY : c.TZ;
  std::vector<vec*> Qs = {&c.pxm, &c.pxp, &c.pym, &c.pyp, &c.pzm, &c.pzp};
  if (c.eos == ORC_ADIABATIC) Qs.push_back(&c.e);
#pragma omp parallel   // OpenMP build only: lines are independent (a line reads and writes only its own cells)
  {
  vec r(n), ir(n), f(n), a(n), fs(n), rs(n), Fr(n), FQ(n), w(n), len(n), invd(n), S(n + 1), dtiv(n);   // line buffers
#pragma omp for collapse(2) schedule(static)
  for (int q = 0; q < Q; ++q)
    for (int p = 0; p < P; ++p) {
      auto L = [&](int m) -> size_t {   // line position (halo-inclusive) -> linear index
        int t = m - H;
        if (wrap) { t %= T; if (t < 0) t += T; }
        return dir == 0 ? c.id(t, p, q) : dir == 1 ? c.id(p, t, q) : c.id(p, q, t);
      };
      // geometry and frozen face velocity along the line (velocities are not updated during transport)
      for (int m = 0; m < n; ++m) {
        int t = m - H; if (wrap) { t %= T; if (t < 0) t += T; }
        int j = dir == 0 ? p : dir == 1 ? t : q;
        int k = dir == 0 ? q : dir == 1 ? q : t;
        if (dir == 0) {
          len[m] = c.LX(j, k); invd[m] = c.invLX(j, k); S[m] = c.Sx(j, k);
          w[m] = c.vx[L(m)] - c.v0[c.rid(j, k)];        // residual velocity with FARGO; v0 = 0 otherwise
        } else if (dir == 1) {
          len[m] = c.LY[j]; invd[m] = c.invDY[j]; S[m] = c.Sy(j, k); w[m] = c.vy[L(m)];
        } else {
          len[m] = c.LZ(j, k); invd[m] = c.invDZ(j, k); S[m] = c.Sz(j, k); w[m] = c.vz[L(m)];
        }
        dtiv[m] = dt * c.invV(j, k);
        r[m] = c.rho[L(m)];
        ir[m] = 1.0 / r[m];
      }
      // density: slope, star value, mass flux F = w rho* S (Eqs. 45-47)
      oracle_vanleer_slopes(n, r.data(), invd.data(), a.data());
      oracle_vanleer_star(n, r.data(), a.data(), len.data(), w.data(), dt, rs.data());
      for (int m = 0; m < n; ++m) Fr[m] = (w[m] * rs[m]) * S[m];
      // every other quantity: q = Q/rho (consistent transport), F_Q = F_rho q*
      for (vec* Qp : Qs) {
        vec& Qa = *Qp;
        for (int m = 0; m < n; ++m) f[m] = Qa[L(m)] * ir[m];
        oracle_vanleer_slopes(n, f.data(), invd.data(), a.data());
        oracle_vanleer_star(n, f.data(), a.data(), len.data(), w.data(), dt, fs.data());
        for (int m = 0; m < n; ++m) FQ[m] = Fr[m] * fs[m];
        for (int m = 2; m + 2 < n; ++m) Qa[L(m)] = std::fma(-dtiv[m], FQ[m + 1] - FQ[m], Qa[L(m)]);
      }
      for (int m = 2; m + 2 < n; ++m) c.rho[L(m)] = std::fma(-dtiv[m], Fr[m + 1] - Fr[m], r[m]);
    }
  }
}

// ---- 12d: new velocities, Eq. 51 with Tab. 2 inverted (reading G28) ----------------------
void orc_newvel(oracle_ctx& c) {
  const double om = (c.geometry == ORC_CARTESIAN) ? 0.0 : c.p.omega_frame;
#pragma omp parallel for collapse(2) schedule(static)   // OpenMP build only: writes v of its own cell, reads momenta and rho
  for (int k = c.k0(); k < c.k1(); ++k)
    for (int j = c.j0(); j < c.j1(); ++j) {
      const double rx = c.Rx(j, k), rx2om = c.shear ? (2.0 * c.p.omega_frame) * c.yc[j] : (rx * rx) * om;
      const double irx = c.invRx(j, k), irz = c.invRzj[j];
      for (int i = c.i0(); i < c.i1(); ++i) {
        const size_t l = c.id(i, j, k);
        if (c.hasx) {
          const size_t lm = c.id(c.xw(i - 1), j, k);
          c.vx[l] = ((c.pxp[lm] + c.pxm[l]) / (c.rho[lm] + c.rho[l]) - rx2om) * irx;
        }
        if (c.hasy) {
          const size_t lm = c.id(i, j - 1, k);
          c.vy[l] = (c.pyp[lm] + c.pym[l]) / (c.rho[lm] + c.rho[l]);
        }
        if (c.hasz) {
          const size_t lm = c.id(i, j, k - 1);
          c.vz[l] = ((c.pzp[lm] + c.pzm[l]) / (c.rho[lm] + c.rho[l])) * irz;
        }
      }
    }
}
