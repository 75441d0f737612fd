// orbital.cpp -- the FARGO orbital-advection step (section 3.5.1): for each ring (j,k) the
// uniform part v0_jk of the azimuthal velocity (Eq. 72) moves the ring by s = v0 dt / LX cells, split
// (Eqs. 65-68) into an integer number of cells N = E(s) (Eq. 66; circular permutation, Eq. 69) and a
// fractional remainder xi = s - N, |xi| <= 1/2, advected conservatively (Eq. 70) with the
// Piecewise Parabolic Advection star values.
// CPU oracle, TEST INFRASTRUCTURE (see fargo_oracle.h).
#include "oracle_impl.hpp"

// ---- 1-D primitives on a periodic ring of n cells ------------------------------------------------
static inline int wrapi(int i, int n) { int m = i % n; return m < 0 ? m + n : m; }

// Monotonised left/right interface values of every cell.
//   dQ_i   = (Q_{i+1} - Q_{i-1})/2
//   dmQ_i  = 0 if (Q_{i+1}-Q_i)(Q_i-Q_{i-1}) <= 0, else sgn(dQ_i) min(2|Q_i-Q_{i-1}|, 2|Q_{i+1}-Q_i|, |dQ_i|)
//   Q^L_{i+1} = Q^R_i = Q_i + (Q_{i+1}-Q_i)/2 - (dmQ_{i+1} - dmQ_i)/6                                       (Eq. 71)
// then the three mutually exclusive final tests of P:484, with Delta_i and C_i evaluated once from the
// un-limited values.
extern "C" void oracle_ppa_interfaces(int n, const double* f, double* fl, double* fr) {
  std::vector<double> dm(n);
  for (int i = 0; i < n; ++i) {
    const double fm = f[wrapi(i - 1, n)], f0 = f[i], fp = f[wrapi(i + 1, n)];
    const double a = f0 - fm, b = fp - f0;
    const double d = 0.5 * (fp - fm);
    if (a * b <= 0.0) dm[i] = 0.0;
    else {
      const double m = std::fmin(std::fmin(2.0 * std::fabs(a), 2.0 * std::fabs(b)), std::fabs(d));
      dm[i] = d < 0.0 ? -m : m;
    }
  }
  for (int i = 0; i < n; ++i) {
    const int ip = wrapi(i + 1, n);
    const double v = std::fma(0.5, f[ip] - f[i], f[i]) - (dm[ip] - dm[i]) / 6.0;
    fr[i] = v;
    fl[ip] = v;
  }
  for (int i = 0; i < n; ++i) {
    const double fm = f[wrapi(i - 1, n)], f0 = f[i], fp = f[wrapi(i + 1, n)];
    const double a = f0 - fm, b = fp - f0;
    if (a * b <= 0.0) { fl[i] = f0; fr[i] = f0; continue; }
    const double D = fr[i] - fl[i];
    const double C = std::fma(-0.5, fl[i] + fr[i], f0);
    const double DC = D * C, D26 = (D * D) / 6.0;
    if (DC > D26) fl[i] = std::fma(3.0, f0, -(2.0 * fr[i]));
    else if (-D26 > DC) fr[i] = std::fma(3.0, f0, -(2.0 * fl[i]));
  }
}

// Star value on face i+1/2 for a uniform displacement of xi cells (formula at P:470; reading G15:
// the branch is chosen by the sign of the velocity, and x = |xi| enters both branches, which makes
// the value the average of the parabola over the swept interval).
extern "C" void oracle_ppa_star(int n, const double* f, double xi, double* fstar) {
  std::vector<double> fl(n), fr(n);
  oracle_ppa_interfaces(n, f, fl.data(), fr.data());
  const double x = std::fabs(xi);
  const double x1x = x * (1.0 - x);
  for (int i = 0; i < n; ++i) {
    const int u = (xi >= 0.0) ? i : wrapi(i + 1, n);   // upwind cell of face i+1/2
    const double edge = (xi >= 0.0) ? fr[u] : fl[u];   // its interface value on that face
    fstar[i] = std::fma(x1x, std::fma(2.0, f[u], -fr[u]) - fl[u], std::fma(x, f[u] - edge, edge));
  }
}

// ---- O10a: fractional uniform sweep (Eq. 70) on rho and on q = Q/rho (reading G17) ---------------
// "Same advection machinery": mass flux through face i+1/2 over dt, per unit of (LX Sx), is
// xi rho*; the flux of Q is that times q*; update as Eqs. 41-43 with dt V^-1 (F_{i+1/2} - F_{i-1/2}),
// where w dt S = xi LX Sx for the ring-uniform velocity w = xi LX / dt.
void orc_orbital_frac(oracle_ctx& c) {
  if (!c.p.fargo_on) return;
  const int n = c.TX;   // FARGO requires wrapped X: TX = nx
  std::vector<vec*> Qs = {&c.pxm, &c.pxp, &c.pym, &c.pyp, &c.pzm, &c.pzp};
  if (c.eos == ORC_ADIABATIC) Qs.push_back(&c.e);
#pragma omp parallel   // OpenMP build only: rings are independent
  {
  vec r(n), ir(n), f(n), rs(n), fs(n), Fr(n), FQ(n);   // ring buffers
#pragma omp for collapse(2) schedule(static)
  for (int k = 0; k < c.TZ; ++k)
    for (int j = 0; j < c.TY; ++j) {
      const double s = (c.v0[c.rid(j, k)] * c.dt) * c.invLX(j, k);
      const double N = std::floor(s + 0.5);             // nearest integer (Eq. 66; reading G11)
      const double xi = s - N;
      c.nshift[c.rid(j, k)] = N;
      c.xi[c.rid(j, k)] = xi;
      const double g = (c.LX(j, k) * c.Sx(j, k)) * c.invV(j, k);
      const size_t base = c.id(0, j, k);
      for (int i = 0; i < n; ++i) { r[i] = c.rho[base + i]; ir[i] = 1.0 / r[i]; }
      oracle_ppa_star(n, r.data(), xi, rs.data());
      for (int i = 0; i < n; ++i) Fr[i] = xi * rs[i];
      for (vec* Qp : Qs) {
        vec& Qa = *Qp;
        for (int i = 0; i < n; ++i) f[i] = Qa[base + i] * ir[i];
        oracle_ppa_star(n, f.data(), xi, fs.data());
        for (int i = 0; i < n; ++i) FQ[i] = Fr[i] * fs[i];
        for (int i = 0; i < n; ++i) Qa[base + i] = std::fma(-g, FQ[i] - FQ[wrapi(i - 1, n)], Qa[base + i]);
      }
      for (int i = 0; i < n; ++i) c.rho[base + i] = std::fma(-g, Fr[i] - Fr[wrapi(i - 1, n)], r[i]);
    }
  }
}

// ---- O10b: integer shift, Q_i <- Q_{i-N} (Eq. 69) ---------------------------------------
void orc_orbital_shift(oracle_ctx& c) {
  if (!c.p.fargo_on) return;
  const int n = c.TX;
  std::vector<vec*> Qs = {&c.rho, &c.pxm, &c.pxp, &c.pym, &c.pyp, &c.pzm, &c.pzp};
  if (c.eos == ORC_ADIABATIC) Qs.push_back(&c.e);
#pragma omp parallel   // OpenMP build only: rings are independent
  {
  vec tmp(n);
#pragma omp for collapse(2) schedule(static)
  for (int k = 0; k < c.TZ; ++k)
    for (int j = 0; j < c.TY; ++j) {
      const long long N = (long long)c.nshift[c.rid(j, k)];
      const int sh = (int)(((N % n) + n) % n);
      if (sh == 0) continue;
      const size_t base = c.id(0, j, k);
      for (vec* Qp : Qs) {
        vec& Qa = *Qp;
        for (int i = 0; i < n; ++i) tmp[i] = Qa[base + wrapi(i - sh, n)];
        for (int i = 0; i < n; ++i) Qa[base + i] = tmp[i];
      }
    }
  }
}
