// k_mhd.cu -- SURVEY.md 8(f) NEXT-4: the MHD substeps of Fig. 2 on 3-D Cartesian meshes (sections 3.6.1-3.6.2):
//   k_bc_b         cell 2    ghost fill of the face-centred field (the normal component keeps its boundary face)
//   k_mhd_pressure cell 7a   gradient of the zone-centred magnetic pressure of the transverse components
//   k_mhd_emf      cells 8a-8c  star values by the method of characteristics (Eqs. 80-83), electromotive forces (Eq. 84),
//                            resistive term, and the "Lagrangian" star values of cell 8d (note 14)
//   k_mhd_tension  cell 8d   magnetic tension on the velocities (Eq. 86)
//   k_mhd_ct       cell 10   constrained transport (Eq. 76 with the signs of Eq. 101; reading G35)
//   k_mhd_resid, k_mhd_arc, k_mhd_orbital   cell 11: orbital advection of B by the upstream-averaged EMF (section 3.7)
// and the Alfven speed for cell 6 (Eq. 59 item 1).  One thread per edge / face, neighbours through L1/L2; the expressions and their order are those of docs/ARITHMETIC.md ("MHD"), so the results agree with the CPU
// oracle to rounding (bit for bit in fp64).  Product code: shares nothing with oracle/.
// Directions 0, 1, 2 = X, Y, Z; (D1, D2, D3) cyclic; eps_D3 = v_D1 B_D2 - v_D2 B_D1 lives on the edge along D3 at the
// lower-D1, lower-D2 corner of its cell; a component along D lives on the lower D face.
#include "kernels.h"

namespace fg {

// a cell and its linear index (kept along by mv: a neighbour costs an addition, not an index product)
template <typename T> struct Cell { int n[3]; long long l; };
template <typename T>
__device__ __forceinline__ Cell<T> cell(const Dev<T>& d, const int i, const int j, const int k) { return Cell<T>{{i, j, k}, d.id(i, j, k)}; }

template <typename T>
__device__ __forceinline__ int ext_of(const Dev<T>& d, const int dir) { return dir == 0 ? d.TX : dir == 1 ? d.TY : d.TZ; }
// the cell s steps along dir (X wraps when periodic)
template <typename T>
__device__ __forceinline__ Cell<T> mv(const Dev<T>& d, Cell<T> q, const int dir, const int s) {
  int m = q.n[dir] + s;
  if (dir == 0 && d.xwrap) { if (m < 0) m += d.nx; else if (m >= d.nx) m -= d.nx; }
  q.l += dir == 0 ? (long long)(m - q.n[0]) : dir == 1 ? s * d.pitch : s * d.plane;
  q.n[dir] = m;
  return q;
}
template <typename T>
__device__ __forceinline__ long long at(const Dev<T>&, const Cell<T>& q) { return q.l; }
// R_x = 1 | r | r sin(theta), R_z = 1 | 1 | r (Tab. 1) where a quantity on the lower f face of cell q sits (f = 1: at the
// lower Y edge, f = 2: at the lower Z edge, else at the zone centre), and their reciprocals (host tables).  On a Cartesian
// mesh every factor is 1.0 and the products below are exact (reading G38).
template <typename T> __device__ __forceinline__ T RxJ(const Dev<T>& d, const Cell<T>& q, const int f) { return d.geometry == GEO_CART ? T(1) : (f == 1 ? d.ye[q.n[1]] : d.yc[q.n[1]]); }
template <typename T> __device__ __forceinline__ T RxK(const Dev<T>& d, const Cell<T>& q, const int f) { return d.geometry == GEO_SPH ? (f == 2 ? d.sin_ze[q.n[2]] : d.sin_zc[q.n[2]]) : T(1); }
template <typename T> __device__ __forceinline__ T RzJ(const Dev<T>& d, const Cell<T>& q, const int f) { return d.geometry == GEO_SPH ? (f == 1 ? d.ye[q.n[1]] : d.yc[q.n[1]]) : T(1); }
template <typename T> __device__ __forceinline__ T iRxJ(const Dev<T>& d, const Cell<T>& q, const int f) { return d.geometry == GEO_CART ? T(1) : (f == 1 ? d.inv_ye[q.n[1]] : d.inv_yc[q.n[1]]); }
template <typename T> __device__ __forceinline__ T iRxK(const Dev<T>& d, const Cell<T>& q, const int f) { return d.geometry == GEO_SPH ? (f == 2 ? d.inv_sin_ze[q.n[2]] : d.invRxk[q.n[2]]) : T(1); }
template <typename T> __device__ __forceinline__ T iRzJ(const Dev<T>& d, const Cell<T>& q, const int f) { return d.geometry == GEO_SPH ? (f == 1 ? d.inv_ye[q.n[1]] : d.inv_yc[q.n[1]]) : T(1); }
// physical width of cell q along dir and 1 / (distance of its centre from the centre below), for a quantity on the lower f face
template <typename T>
__device__ __forceinline__ T width(const Dev<T>& d, const int dir, const Cell<T>& q, const int f) {
  return dir == 0 ? (d.dx * RxJ(d, q, f)) * RxK(d, q, f) : dir == 1 ? d.LY[q.n[1]] : d.dz[q.n[2]] * RzJ(d, q, f);
}
template <typename T>
__device__ __forceinline__ T invdist(const Dev<T>& d, const int dir, const Cell<T>& q, const int f) {
  return dir == 0 ? (d.invdx * iRxJ(d, q, f)) * iRxK(d, q, f) : dir == 1 ? d.invDY[q.n[1]] : d.invdzc[q.n[2]] * iRzJ(d, q, f);
}
template <typename T>
__device__ __forceinline__ bool fits(const Dev<T>& d, const int dir, const int n, const int lo, const int hi) {
  if (dir == 0 && d.xwrap) return true;
  return n - lo >= 0 && n + hi < ext_of(d, dir);
}

// The linear reconstructions of f in the two zones next to the lower dir face of cell q: every star value on that face
// (upwind estimate, the two feet of the characteristics, the Lagrangian ones: five per field) picks one of the two, so the
// slopes -- a division each -- are formed once per field and face instead of once per star value.
template <typename T> struct Recon {
  T fm, f0, sm, s0, wm, w0;
  __device__ __forceinline__ T star(const T w, const T dt) const {   // Eq. 48
    return w >= T(0) ? rfma(sm, rfma(-w, dt, wm) * T(0.5), fm) : rfma(-s0, rfma(w, dt, w0) * T(0.5), f0);
  }
};
template <typename T>   // van Leer slope
__device__ __forceinline__ T slope3(const T fm, const T f0, const T fp, const T invd0, const T invdp) {
  const T dm = (f0 - fm) * invd0, dp = (fp - f0) * invdp;
  const T pr = dm * dp;
  const bool flat = pr <= T(0);
  const T a = rdiv(T(2) * pr, flat ? T(1) : dm + dp);
  return flat ? T(0) : a;
}
template <typename T>   // fc: the direction of the faces f lives on (it fixes the lengths on a curvilinear mesh)
__device__ __forceinline__ Recon<T> recon(const Dev<T>& d, const T* __restrict__ f, const Cell<T>& q, const int dir, const int fc) {
  const Cell<T> qm = mv(d, q, dir, -1), qp = mv(d, q, dir, +1);
  const T f2 = f[at(d, mv(d, qm, dir, -1))], f1 = f[at(d, qm)], f0 = f[at(d, q)], fp = f[at(d, qp)];
  const T im = invdist(d, dir, dir == 0 ? q : qm, fc), i0 = invdist(d, dir, q, fc), ip = invdist(d, dir, dir == 0 ? q : qp, fc);
  Recon<T> r;
  r.fm = f1; r.f0 = f0;
  r.sm = slope3(f2, f1, f0, im, i0);
  r.s0 = slope3(f1, f0, fp, i0, ip);
  r.wm = width(d, dir, qm, fc); r.w0 = width(d, dir, q, fc);
  return r;
}

template <typename T> struct Vec3 { T* c[3]; };
template <typename T> __global__ void k_mhd_curv(const Dev<T> d, const T* __restrict__ rho, const Vec3<T> b, const Vec3<T> vb, const T mu0);

// ---- cell 2 ------------------------------------------------------------------------------------------------------------
template <typename T, int DIR>
__global__ void k_bc_b(const Dev<T> d, const Vec3<T> b) {
  if (d.ctl->done) return;
  const int N = DIR == 0 ? d.nx : DIR == 1 ? d.ny : d.nz;
  const int ng = DIR == 0 ? d.ngx : DIR == 1 ? d.ngy : d.ngz;
  const int P = DIR == 0 ? d.TY : d.TX, Q = DIR == 2 ? d.TY : d.TZ;
  const int p = blockIdx.x * blockDim.x + threadIdx.x, q = blockIdx.y;
  if (p >= P || q >= Q) return;
  const long long base = DIR == 0 ? d.id(0, p, q) : DIR == 1 ? d.id(p, 0, q) : d.id(p, q, 0);
  const long long str = DIR == 0 ? 1 : DIR == 1 ? d.pitch : d.plane;
  const int m0 = ng, m1 = ng + N, lo = d.bc[DIR][0], hi = d.bc[DIR][1];
#pragma unroll
  for (int f = 0; f < 3; ++f) {
    T* a = b.c[f] + base;
    const bool normal = f == DIR;
    for (int g = 0; g < ng; ++g) {
      if (lo == BC_PERIODIC) a[(m0 - 1 - g) * str] = a[(m1 - 1 - g) * str];
      else if (lo == BC_OUTFLOW) a[(m0 - 1 - g) * str] = a[m0 * str];
      else a[(m0 - 1 - g) * str] = normal ? a[(m0 + 1 + g) * str] : a[(m0 + g) * str];
      if (hi == BC_PERIODIC) a[(m1 + g) * str] = a[(m0 + g) * str];
      else if (normal) { if (g >= 1) a[(m1 + g) * str] = hi == BC_OUTFLOW ? a[m1 * str] : a[(m1 - g) * str]; }
      else a[(m1 + g) * str] = hi == BC_OUTFLOW ? a[(m1 - 1) * str] : a[(m1 - 1 - g) * str];
    }
  }
}

template <typename T>
int launch_bc_b(const Dev<T>& d, T* bx, T* by, T* bz, cudaStream_t s) {
  Vec3<T> b{{bx, by, bz}};
  int n = 0;
  if (d.ngx > 0) { k_bc_b<T, 0><<<dim3((d.TY + 63) / 64, d.TZ), 64, 0, s>>>(d, b); ++n; }
  if (d.ngy > 0) { k_bc_b<T, 1><<<dim3((d.TX + 127) / 128, d.TZ), 128, 0, s>>>(d, b); ++n; }
  if (d.ngz > 0) { k_bc_b<T, 2><<<dim3((d.TX + 127) / 128, d.TY), 128, 0, s>>>(d, b); ++n; }
  return n;
}

// ---- cell 7a: v_b -= dt * 2 / (rho + rho_-) * (Pm - Pm_-) / Delta, Pm = (B_a^2 + B_b^2) / (2 mu0) at the zone centre ------
template <typename T>
__device__ __forceinline__ T pmag(const Dev<T>& d, const Vec3<T>& b, const Cell<T>& q, const int dir, const T mu0) {
  T s = T(0);
#pragma unroll
  for (int t = 1; t <= 2; ++t) {
    const int a = (dir + t) % 3;
    const T bc = T(0.5) * (b.c[a][at(d, q)] + b.c[a][at(d, mv(d, q, a, +1))]);
    s = rfma(bc, bc, s);
  }
  return rdiv(s, T(2) * mu0);
}
template <typename T, int GEO>
__global__ void __launch_bounds__(128, 16) k_mhd_pressure(const Dev<T> d_in, const T* __restrict__ rho, const Vec3<T> b, const Vec3<T> vb, const T mu0) {
  Dev<T> d = d_in;
  if (GEO == GEO_CART) d.geometry = GEO_CART;
  if (d.ctl->done) return;
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= d.TX) return;
  const Cell<T> q = cell(d, i, (int)blockIdx.y, (int)blockIdx.z);
  const T dt = (T)d.ctl->dt;
#pragma unroll
  for (int dir = 0; dir < 3; ++dir) {
    const int da = (dir + 1) % 3, db = (dir + 2) % 3;
    if (!fits(d, dir, q.n[dir], 1, 0) || !fits(d, da, q.n[da], 0, 1) || !fits(d, db, q.n[db], 0, 1)) continue;
    const Cell<T> qm = mv(d, q, dir, -1);
    const long long l = at(d, q);
    // as 7a's pressure gradient (on a Cartesian mesh invLX = 1/dx and invDZ = invdzc: the table factors are 1.0)
    const T il = GEO == GEO_CART ? (dir == 0 ? d.invdx : dir == 1 ? d.invDY[q.n[1]] : d.invdzc[q.n[2]])
                                 : (dir == 0 ? d.invLX(q.n[1], q.n[2]) : dir == 1 ? d.invDY[q.n[1]] : d.invDZ(q.n[1], q.n[2]));
    const T wf = rdiv(T(2) * il, rho[l] + rho[at(d, qm)]);
    vb.c[dir][l] = rfma(-dt, wf * (pmag(d, b, q, dir, mu0) - pmag(d, b, qm, dir, mu0)), vb.c[dir][l]);
  }
}
template <typename T>
int launch_mhd_pressure(const Dev<T>& d, const T* rho, T* bx, T* by, T* bz, T* vxb, T* vyb, T* vzb, double mu0, cudaStream_t s) {
  const dim3 g((d.TX + 127) / 128, d.TY, d.TZ);
  if (d.geometry == GEO_CART) { k_mhd_pressure<T, GEO_CART><<<g, 128, 0, s>>>(d, rho, Vec3<T>{{bx, by, bz}}, Vec3<T>{{vxb, vyb, vzb}}, (T)mu0); return 1; }
  k_mhd_pressure<T, GEO_CYL><<<g, 128, 0, s>>>(d, rho, Vec3<T>{{bx, by, bz}}, Vec3<T>{{vxb, vyb, vzb}}, (T)mu0);   // (any curvilinear tag: tables are read)
  k_mhd_curv<T><<<dim3((d.TX + 127) / 128, d.TY, d.TZ), 128, 0, s>>>(d, rho, Vec3<T>{{bx, by, bz}}, Vec3<T>{{vxb, vyb, vzb}}, (T)mu0);
  return 2;
}

// ---- cells 8a-8c (+ the star values of 8d): one thread per edge along D3 ----------------------------------------------
// GEO is the mesh geometry as a compile-time constant: on a Cartesian mesh every metric factor folds to 1.0 and its table
// loads disappear (the run-time test cost a third of the kernel's time at 512^3)
template <typename T, int D3, int GEO>
__global__ void __launch_bounds__(128) k_mhd_emf(const Dev<T> d_in, const T* __restrict__ rho, const Vec3<T> v, const Vec3<T> b,
                                                 T* __restrict__ E, T* __restrict__ S1, T* __restrict__ S2, const T mu0, const T eta) {
  constexpr int D1 = (D3 + 1) % 3, D2 = (D3 + 2) % 3;
  Dev<T> d = d_in;
  d.geometry = GEO;
  if (d.ctl->done) return;
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= d.TX) return;
  const Cell<T> q = cell(d, i, (int)blockIdx.y, (int)blockIdx.z);
  const long long l = at(d, q);
  const T* __restrict__ V1 = v.c[D1];
  const T* __restrict__ V2 = v.c[D2];
  const T* __restrict__ B1 = b.c[D1];
  const T* __restrict__ B2 = b.c[D2];
  if (!fits(d, D1, q.n[D1], 2, 1) || !fits(d, D2, q.n[D2], 2, 1)) { E[l] = T(0); S1[l] = B1[l]; S2[l] = B2[l]; return; }
  const T dt = (T)d.ctl->dt;
  const Cell<T> q1 = mv(d, q, D1, -1), q2 = mv(d, q, D2, -1), q12 = mv(d, q1, D2, -1);
  const long long l1 = at(d, q1), l2 = at(d, q2);
  // density at the edge: the four zones around it
  const T ro = T(0.25) * (((rho[l] + rho[l1]) + rho[l2]) + rho[at(d, q12)]);
  const T sr = rsqrt_ieee(mu0 * ro);
  // the reconstructions every star value on this edge picks from: (v_D1, B_D1) along D2, (v_D2, B_D2) along D1
  const Recon<T> rV1 = recon(d, V1, q, D2, D1), rB1 = recon(d, B1, q, D2, D1), rV2 = recon(d, V2, q, D1, D2), rB2 = recon(d, B2, q, D1, D2);
  // upwind estimates of the transverse fields (superscript u)
  const T v2bar = T(0.5) * (V2[l] + V2[l1]);
  const T v1bar = T(0.5) * (V1[l] + V1[l2]);
  const T v1u = rV1.star(v2bar, dt), B1u = rB1.star(v2bar, dt);
  const T v2u = rV2.star(v1bar, dt), B2u = rB2.star(v1bar, dt);
  T v2s, B2s, v1s, B1s;
  {   // (v_D2*, B_D2*): 1.5-D problem along D1 (Eqs. 80-83)
    const T a = rdiv(B1u, sr);
    const T Cp = v1u - a, Cm = v1u + a;
    const T vp = rV2.star(Cp, dt), Bp = rB2.star(Cp, dt), vm = rV2.star(Cm, dt), Bm = rB2.star(Cm, dt);
    v2s = T(0.5) * ((vp + vm) + rdiv(Bp - Bm, sr));
    B2s = T(0.5) * ((Bp + Bm) + sr * (vp - vm));
  }
  {   // (v_D1*, B_D1*): 1.5-D problem along D2
    const T a = rdiv(B2u, sr);
    const T Cp = v2u - a, Cm = v2u + a;
    const T vp = rV1.star(Cp, dt), Bp = rB1.star(Cp, dt), vm = rV1.star(Cm, dt), Bm = rB1.star(Cm, dt);
    v1s = T(0.5) * ((vp + vm) + rdiv(Bp - Bm, sr));
    B1s = T(0.5) * ((Bp + Bm) + sr * (vp - vm));
  }
  T emf = T(0.5) * (((v1s * B2u + B2s * v1u) - v2s * B1u) - B1s * v2u);   // Eq. 84
  if (eta != T(0)) {   // cell 8c: - eta (curl B)_D3
    T J = (B2[l] - B2[l1]) * invdist(d, D1, q, D2);
    J = J - (B1[l] - B1[l2]) * invdist(d, D2, q, D1);
    emf = rfma(-eta, J, emf);
  }
  E[l] = emf;
  {   // cell 8d star values: characteristic speeds -+ B / sqrt(mu0 rho) only
    const T a = rdiv(T(0.5) * (B2[l] + B2[l1]), sr);
    const T vp = rV1.star(-a, dt), Bp = rB1.star(-a, dt), vm = rV1.star(a, dt), Bm = rB1.star(a, dt);
    S1[l] = T(0.5) * ((Bp + Bm) + sr * (vp - vm));
  }
  {
    const T a = rdiv(T(0.5) * (B1[l] + B1[l2]), sr);
    const T vp = rV2.star(-a, dt), Bp = rB2.star(-a, dt), vm = rV2.star(a, dt), Bm = rB2.star(a, dt);
    S2[l] = T(0.5) * ((Bp + Bm) + sr * (vp - vm));
  }
}

template <typename T>
int launch_mhd_emf(const Dev<T>& d, const T* rho, T* vx, T* vy, T* vz, T* bx, T* by, T* bz, T* const* emf, T* const* bstar,
                   double mu0, double eta, cudaStream_t s) {
  const Vec3<T> v{{vx, vy, vz}}, b{{bx, by, bz}};
  dim3 g((d.TX + 127) / 128, d.TY, d.TZ);
#define FG_EMF(GEO)                                                                                     \
  k_mhd_emf<T, 0, GEO><<<g, 128, 0, s>>>(d, rho, v, b, emf[0], bstar[0], bstar[1], (T)mu0, (T)eta);      \
  k_mhd_emf<T, 1, GEO><<<g, 128, 0, s>>>(d, rho, v, b, emf[1], bstar[2], bstar[3], (T)mu0, (T)eta);      \
  k_mhd_emf<T, 2, GEO><<<g, 128, 0, s>>>(d, rho, v, b, emf[2], bstar[4], bstar[5], (T)mu0, (T)eta);
  if (d.geometry == GEO_CART) { FG_EMF(GEO_CART) }
  else if (d.geometry == GEO_CYL) { FG_EMF(GEO_CYL) }
  else { FG_EMF(GEO_SPH) }
#undef FG_EMF
  return 3;
}

// ---- cell 8d: Eq. 86; cell 10: Eq. 76 ---------------------------------------------------------------------------------------
// bstar[2 D3 + 0] = B_D1* and bstar[2 D3 + 1] = B_D2* on the edges along D3.  For v_D (D, DA, DB cyclic): B_D* on the edges
// along DB is bstar[2 DB + 0] (there D1 = D), on the edges along DA it is bstar[2 DA + 1] (there D2 = D).
template <typename T>
struct MhdArrays { const T* b[3]; const T* emf[3]; const T* bstar[6]; };

template <typename T, bool CART>
__global__ void __launch_bounds__(128, 16) k_mhd_tension(const Dev<T> d_in, const T* __restrict__ rho, const MhdArrays<T> A, const Vec3<T> v, const T mu0) {
  Dev<T> d = d_in;
  if (CART) d.geometry = GEO_CART;
  if (d.ctl->done) return;
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= d.TX) return;
  const Cell<T> q = cell(d, i, (int)blockIdx.y, (int)blockIdx.z);
  const long long l = at(d, q);
  const T dt = (T)d.ctl->dt;
#pragma unroll
  for (int D = 0; D < 3; ++D) {
    const int DA = (D + 1) % 3, DB = (D + 2) % 3;
    if (!fits(d, D, q.n[D], 2, 1) || !fits(d, DA, q.n[DA], 2, 2) || !fits(d, DB, q.n[DB], 2, 2)) continue;
    const T* __restrict__ Ba = A.b[DA];
    const T* __restrict__ Bb = A.b[DB];
    const T* __restrict__ Sa = A.bstar[2 * DB + 0];
    const T* __restrict__ Sb = A.bstar[2 * DA + 1];
    const Cell<T> qm = mv(d, q, D, -1), qa = mv(d, q, DA, +1), qb = mv(d, q, DB, +1);
    const long long lm = at(d, qm), la = at(d, qa), lb = at(d, qb);
    const T Bbar_a = T(0.25) * (((Ba[l] + Ba[la]) + Ba[lm]) + Ba[at(d, mv(d, qm, DA, +1))]);
    const T Bbar_b = T(0.25) * (((Bb[l] + Bb[lb]) + Bb[lm]) + Bb[at(d, mv(d, qm, DB, +1))]);
    T acc = Bbar_a * rdiv(Sa[la] - Sa[l], width(d, DA, q, D));
    acc = rfma(Bbar_b, rdiv(Sb[lb] - Sb[l], width(d, DB, q, D)), acc);
    const T wf = rdiv(T(2), mu0 * (rho[l] + rho[lm]));
    v.c[D][l] = rfma(dt, wf * acc, v.c[D][l]);
  }
}

template <typename T, bool CART>
__global__ void __launch_bounds__(128, 16) k_mhd_ct(const Dev<T> d_in, const MhdArrays<T> A, const Vec3<T> b) {
  Dev<T> d = d_in;
  if (CART) d.geometry = GEO_CART;
  if (d.ctl->done) return;
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= d.TX) return;
  const Cell<T> q = cell(d, i, (int)blockIdx.y, (int)blockIdx.z);
  const long long l = at(d, q);
  const T dt = (T)d.ctl->dt;
  if (d.geometry != GEO_CART) {
    // Eq. 76 proper: d(B S)/dt = circulation of eps around the face with the physical edge lengths, over Tab. 5's area:
    // Z edge at (i-1/2, j-1/2, k): lZ = dz R_z(edge j); X edge at (i, j-1/2, k-1/2): lX = dx R_x(edge j, edge k); Y edge: LY[j]
    const int j = q.n[1], k = q.n[2];
    const bool sph = d.geometry == GEO_SPH;
    auto lZ = [&](const int jj) { return d.dz[k] * (sph ? d.ye[jj] : T(1)); };
    auto lX = [&](const int jj, const int kk) { return (d.dx * d.ye[jj]) * (sph ? d.sin_ze[kk] : T(1)); };
    const long long li = at(d, mv(d, q, 0, +1)), lj = l + d.pitch, lk = l + d.plane;
    const T* __restrict__ EX = A.emf[0];
    const T* __restrict__ EY = A.emf[1];
    const T* __restrict__ EZ = A.emf[2];
    if (fits(d, 0, i, 2, 1) && fits(d, 1, j, 2, 2) && fits(d, 2, k, 2, 2)) {
      T circ = EZ[lj] * lZ(j + 1) - EZ[l] * lZ(j);
      circ = circ - (EY[lk] - EY[l]) * d.LY[j];
      b.c[0][l] = rfma(dt, rdiv(circ, d.Sx(j, k)), b.c[0][l]);
    }
    if (fits(d, 1, j, 2, 1) && fits(d, 2, k, 2, 2) && fits(d, 0, i, 2, 2)) {
      T circ = EX[lk] * lX(j, k + 1) - EX[l] * lX(j, k);
      circ = circ - (EZ[li] - EZ[l]) * lZ(j);
      b.c[1][l] = rfma(dt, rdiv(circ, d.Sy(j, k)), b.c[1][l]);
    }
    if (fits(d, 2, k, 2, 1) && fits(d, 0, i, 2, 2) && fits(d, 1, j, 2, 2)) {
      T circ = (EY[li] - EY[l]) * d.LY[j];
      circ = circ - (EX[lj] * lX(j + 1, k) - EX[l] * lX(j, k));
      b.c[2][l] = rfma(dt, rdiv(circ, d.Sz(j, k)), b.c[2][l]);
    }
    return;
  }
#pragma unroll
  for (int D = 0; D < 3; ++D) {
    const int DA = (D + 1) % 3, DB = (D + 2) % 3;
    if (!fits(d, D, q.n[D], 2, 1) || !fits(d, DA, q.n[DA], 2, 2) || !fits(d, DB, q.n[DB], 2, 2)) continue;
    const T* __restrict__ Eb = A.emf[DB];
    const T* __restrict__ Ea = A.emf[DA];
    T curl = rdiv(Eb[at(d, mv(d, q, DA, +1))] - Eb[l], width(d, DA, q, D));
    curl = curl - rdiv(Ea[at(d, mv(d, q, DB, +1))] - Ea[l], width(d, DB, q, D));
    b.c[D][l] = rfma(dt, curl, b.c[D][l]);
  }
}

// ---- cell 7a, geometric terms of B.grad B on curvilinear meshes (Eqs. 87-91), applied to v_b in place --------------------
template <typename T>
__device__ __forceinline__ T avg4(const Dev<T>& d, const T* __restrict__ b, const Cell<T>& q, const int da, const int db) {
  const Cell<T> qm = mv(d, q, db, -1);
  return T(0.25) * (((b[at(d, q)] + b[at(d, mv(d, q, da, +1))]) + b[at(d, qm)]) + b[at(d, mv(d, qm, da, +1))]);
}
template <typename T>
__global__ void __launch_bounds__(128) k_mhd_curv(const Dev<T> d, const T* __restrict__ rho, const Vec3<T> b, const Vec3<T> vb, const T mu0) {
  if (d.ctl->done) return;
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= d.TX) return;
  const int j = blockIdx.y, k = blockIdx.z;
  const Cell<T> q = cell(d, i, j, k);
  const long long l = at(d, q);
  const bool sph = d.geometry == GEO_SPH;
  const T dt = (T)d.ctl->dt, imu = rdiv(T(1), mu0);
  const bool zok = !sph || fits(d, 2, k, 1, 1);
  // all three read B only: the in-place update of v_b is safe
  if (fits(d, 0, i, 1, 0) && fits(d, 1, j, 0, 1) && zok) {   // v_phi: Eqs. 87, 89
    const T wf = rdiv(T(2) * imu, rho[l] + rho[at(d, mv(d, q, 0, -1))]);
    const T bphi = b.c[0][l], br = avg4(d, b.c[1], q, 1, 0);
    T g = br * bphi;
    if (sph) g = rfma(avg4(d, b.c[2], q, 2, 0) * bphi, d.cot_zc[k], g);
    vb.c[0][l] = rfma(dt, (wf * g) * d.inv_yc[j], vb.c[0][l]);
  }
  if (fits(d, 1, j, 1, 0) && fits(d, 0, i, 0, 1) && zok) {    // v_r: Eqs. 88, 90
    const T wf = rdiv(T(2) * imu, rho[l] + rho[at(d, mv(d, q, 1, -1))]);
    const T bphi = avg4(d, b.c[0], q, 0, 1);
    T g = bphi * bphi;
    if (sph) { const T bth = avg4(d, b.c[2], q, 2, 1); g = rfma(bth, bth, g); }
    vb.c[1][l] = rfma(-dt, (wf * g) * d.inv_ye[j], vb.c[1][l]);
  }
  if (sph && fits(d, 2, k, 1, 0) && fits(d, 0, i, 0, 1) && fits(d, 1, j, 0, 1)) {   // v_theta: Eq. 91
    const T wf = rdiv(T(2) * imu, rho[l] + rho[at(d, mv(d, q, 2, -1))]);
    const T bth = b.c[2][l], br = avg4(d, b.c[1], q, 1, 2), bphi = avg4(d, b.c[0], q, 0, 2);
    const T g = rfma(-(bphi * bphi), d.cot_ze[k], br * bth);
    vb.c[2][l] = rfma(dt, (wf * g) * d.inv_yc[j], vb.c[2][l]);
  }
}

template <typename T>
int launch_mhd_tension(const Dev<T>& d, const T* rho, T* const* b, T* const* bstar, T* vx, T* vy, T* vz, double mu0, cudaStream_t s) {
  MhdArrays<T> A;
  for (int n = 0; n < 3; ++n) { A.b[n] = b[n]; A.emf[n] = nullptr; }
  for (int n = 0; n < 6; ++n) A.bstar[n] = bstar[n];
  if (d.geometry == GEO_CART) k_mhd_tension<T, true><<<dim3((d.TX + 127) / 128, d.TY, d.TZ), 128, 0, s>>>(d, rho, A, Vec3<T>{{vx, vy, vz}}, (T)mu0);
  else k_mhd_tension<T, false><<<dim3((d.TX + 127) / 128, d.TY, d.TZ), 128, 0, s>>>(d, rho, A, Vec3<T>{{vx, vy, vz}}, (T)mu0);
  return 1;
}
template <typename T>
int launch_mhd_ct(const Dev<T>& d, T* const* emf, T* bx, T* by, T* bz, cudaStream_t s) {
  MhdArrays<T> A;
  for (int n = 0; n < 3; ++n) { A.b[n] = nullptr; A.emf[n] = emf[n]; }
  for (int n = 0; n < 6; ++n) A.bstar[n] = nullptr;
  if (d.geometry == GEO_CART) k_mhd_ct<T, true><<<dim3((d.TX + 127) / 128, d.TY, d.TZ), 128, 0, s>>>(d, A, Vec3<T>{{bx, by, bz}});
  else k_mhd_ct<T, false><<<dim3((d.TX + 127) / 128, d.TY, d.TZ), 128, 0, s>>>(d, A, Vec3<T>{{bx, by, bz}});
  return 1;
}

// ---- cell 11: orbital advection of B (section 3.7, Eqs. 92-107) -------------------------------------------------------------
// With orbital advection the substeps of cell 8 see the residual velocity v_X - v0 (reading G37).
template <typename T>
__global__ void __launch_bounds__(128) k_mhd_resid(const Dev<T> d, const T* __restrict__ vx, const T* __restrict__ v0, T* __restrict__ vres) {
  if (d.ctl->done) return;
  const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y, k = blockIdx.z;
  if (i >= d.TX) return;
  const long long l = d.id(i, j, k);
  vres[l] = vx[l] - v0[d.rid(j, k)];
}

// Monotonised parabola of zone u of a periodic row: its left and right interface values
template <typename T>
__device__ __forceinline__ T ppa_dm(const T fm, const T f0, const T fp) {
  const T a = f0 - fm, b = fp - f0, dd = T(0.5) * (fp - fm);
  if (a * b <= T(0)) return T(0);
  const T m = rmin(rmin(T(2) * rabs(a), T(2) * rabs(b)), rabs(dd));
  return dd < T(0) ? -m : m;
}
template <typename T>
__device__ __forceinline__ void ppa_zone(const T f2m, const T f1m, const T f0, const T f1p, const T f2p, T& fl, T& fr) {
  const T dmm = ppa_dm(f2m, f1m, f0), dm0 = ppa_dm(f1m, f0, f1p), dmp = ppa_dm(f0, f1p, f2p);
  fr = rfma(T(0.5), f1p - f0, f0) - rdiv6(dmp - dm0);      // Eq. 71
  fl = rfma(T(0.5), f0 - f1m, f1m) - rdiv6(dm0 - dmm);
  const T a = f0 - f1m, b = f1p - f0;
  if (a * b <= T(0)) { fl = f0; fr = f0; return; }
  const T D = fr - fl;
  const T C = rfma(T(-0.5), fl + fr, f0);
  const T DC = D * C, D26 = rdiv6(D * D);
  if (DC > D26) fl = rfma(T(3), f0, -(T(2) * fr));
  else if (-D26 > DC) fr = rfma(T(3), f0, -(T(2) * fl));
}
// (integral of g over the arc of s zones upstream of the face i-1/2) / DX, g a periodic row of n zones (Eq. 96):
// the whole zones one after the other, then the residual fraction from the parabola of the zone it falls in
template <typename T>
__device__ __forceinline__ T arc_integral(const T* __restrict__ g, const int n, const int i, const T s) {
  const T N = floor(s + T(0.5)), xi = s - N;
  const int Ni = (int)N;
  auto w = [n](int m) { m %= n; return m < 0 ? m + n : m; };
  const int c = w(i - 1 - Ni);                         // the star value sits on the face c+1/2
  const int u = xi >= T(0) ? c : w(c + 1);             // its upwind zone
  T fl, fr;
  const T fu = g[u];
  ppa_zone(g[w(u - 2)], g[w(u - 1)], fu, g[w(u + 1)], g[w(u + 2)], fl, fr);
  const T x = rabs(xi), x1x = x * (T(1) - x);
  const T edge = xi >= T(0) ? fr : fl;
  const T gs = rfma(x1x, rfma(T(2), fu, -fr) - fl, rfma(x, fu - edge, edge));
  T S = T(0);
  if (Ni > 0) for (int m = 0; m < Ni; ++m) S = S + g[w(i - 1 - m)];
  if (Ni < 0) for (int m = 1; m <= -Ni; ++m) S = S - g[w(i - 1 + m)];
  return rfma(xi, gs, S);
}
template <typename T>
__global__ void __launch_bounds__(128) k_mhd_arc(const Dev<T> d, const T* __restrict__ by, const T* __restrict__ bz,
                                                 const T* __restrict__ v0, T* __restrict__ PZ, T* __restrict__ PY) {
  if (d.ctl->done) return;
  const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y, k = blockIdx.z;
  if (i >= d.TX) return;
  const long long row = d.id(0, j, k), l = row + i;
  const T dt = (T)d.ctl->dt;
  T pz = T(0), py = T(0);
  if (j >= 1) {   // Z edges of the Y face j-1/2: it moves with the mean of the rings j-1 and j
    const T v0f = T(0.5) * (v0[d.rid(j, k)] + v0[d.rid(j - 1, k)]);
    pz = arc_integral(by + row, d.nx, i, (v0f * dt) * invdist(d, 0, cell(d, 0, j, k), 1));   // zones of the face's own arc length
  }
  if (k >= 1) {   // Y edges of the Z face k-1/2
    const T v0f = T(0.5) * (v0[d.rid(j, k)] + v0[d.rid(j, k - 1)]);
    py = arc_integral(bz + row, d.nx, i, (v0f * dt) * invdist(d, 0, cell(d, 0, j, k), 2));
  }
  PZ[l] = pz; PY[l] = py;
}
template <typename T>
__global__ void __launch_bounds__(128) k_mhd_orbital(const Dev<T> d, const T* __restrict__ PZ, const T* __restrict__ PY, const Vec3<T> b) {
  if (d.ctl->done) return;
  const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y, k = blockIdx.z;
  if (i >= d.TX || j < 1 || j + 1 >= d.TY || k < 1 || k + 1 >= d.TZ) return;
  const long long l = d.id(i, j, k), lp = d.id(d.xw(i + 1), j, k);
  T dd;
  if (d.geometry == GEO_CART) {
    dd = rdiv(d.dx * (PZ[l + d.pitch] - PZ[l]), d.LY[j]);              // Eq. 104 ...
    dd = dd + rdiv(d.dx * (PY[l + d.plane] - PY[l]), d.dz[k]);          // ... and its Z counterpart
  } else {   // cylindrical: the same circulation with each edge's own arc length (Eq. 105), over the area of the face
    const Cell<T> q = cell(d, i, j, k), qj = cell(d, i, j + 1, k), qk = cell(d, i, j, k + 1);
    dd = (width(d, 0, qj, 1) * PZ[l + d.pitch]) * d.dz[k] - (width(d, 0, q, 1) * PZ[l]) * d.dz[k];
    dd = dd + (width(d, 0, qk, 2) * PY[l + d.plane] - width(d, 0, q, 2) * PY[l]) * d.LY[j];
    dd = rdiv(dd, d.Sx(j, k));
  }
  b.c[0][l] = b.c[0][l] + dd;
  b.c[1][l] = b.c[1][l] - (PZ[lp] - PZ[l]);                             // Eq. 101
  b.c[2][l] = b.c[2][l] - (PY[lp] - PY[l]);
}
template <typename T>
int launch_mhd_resid(const Dev<T>& d, const T* vx, const T* v0, T* vres, cudaStream_t s) {
  k_mhd_resid<T><<<dim3((d.TX + 127) / 128, d.TY, d.TZ), 128, 0, s>>>(d, vx, v0, vres);
  return 1;
}
template <typename T>
int launch_mhd_orbital(const Dev<T>& d, const T* v0, T* bx, T* by, T* bz, T* PZ, T* PY, cudaStream_t s) {
  dim3 g((d.TX + 127) / 128, d.TY, d.TZ);
  k_mhd_arc<T><<<g, 128, 0, s>>>(d, by, bz, v0, PZ, PY);
  k_mhd_orbital<T><<<g, 128, 0, s>>>(d, PZ, PY, Vec3<T>{{bx, by, bz}});
  return 2;
}

#define INST(T)                                                                                                          \
  template int launch_mhd_resid<T>(const Dev<T>&, const T*, const T*, T*, cudaStream_t);                                 \
  template int launch_mhd_orbital<T>(const Dev<T>&, const T*, T*, T*, T*, T*, T*, cudaStream_t);                         \
  template int launch_bc_b<T>(const Dev<T>&, T*, T*, T*, cudaStream_t);                                                  \
  template int launch_mhd_pressure<T>(const Dev<T>&, const T*, T*, T*, T*, T*, T*, T*, double, cudaStream_t);            \
  template int launch_mhd_emf<T>(const Dev<T>&, const T*, T*, T*, T*, T*, T*, T*, T* const*, T* const*, double, double, cudaStream_t); \
  template int launch_mhd_tension<T>(const Dev<T>&, const T*, T* const*, T* const*, T*, T*, T*, double, cudaStream_t);   \
  template int launch_mhd_ct<T>(const Dev<T>&, T* const*, T*, T*, T*, cudaStream_t);
INST(double)
INST(float)
#undef INST

}  // namespace fg
