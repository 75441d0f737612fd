// k_source.cu -- the operator-split source step, box 7 of Fig. 2:
//   7a pressure gradient + potential gradient + centrifugal terms (Eqs. 27, 32-38 P:245-280; Eq. 53)
//   7b von Neumann-Richtmyer artificial viscosity, component-wise (readings G8, G19)
//   7c compression work on the energy, time-centred gamma-law form
//   7d viscous stress tensor and force, 2-D cylindrical (App. B, Eqs. B2, B5 P:1202)
// One thread per cell over the whole allocated array; where a stencil would leave the array the input
// is passed through (those cells are re-filled by the ghost fill of cell 9).
#include "kernels.h"

namespace fg {

template <typename T>
__device__ __forceinline__ T pressure(const Dev<T>& d, const T* __restrict__ rho, const T* __restrict__ e, long long l) {
  return d.eos == EOS_ADI ? d.gm1 * e[l] : (e[l] * e[l]) * rho[l];   // Eq. 7 | Eq. 6
}

// ---- 7a ---------------------------------------------------------------------------------------------
template <typename T>
__global__ void __launch_bounds__(128) k_source_a(const Dev<T> d, const State<T> st, const T* __restrict__ phi,
                                                  T* __restrict__ vxb, T* __restrict__ vyb, T* __restrict__ vzb) {
  if (d.ctl->done) return;
  const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y, k = blockIdx.z;
  if (i >= d.TX) return;
  const T dt = (T)d.ctl->dt, om = d.omega;
  const bool curv = d.geometry != GEO_CART, sph = d.geometry == GEO_SPH;
  const long long l = d.id(i, j, k);
  const bool ipok = d.xwrap || i + 1 < d.TX;
  const int ip = d.xw(i + 1);
  const T* __restrict__ rho = st.rho;
  const T* __restrict__ e = st.e;
  const T* __restrict__ vx = st.vx;
  const T* __restrict__ vy = st.vy;
  const T* __restrict__ vz = st.vz;
  const T r0 = rho[l], p0 = pressure(d, rho, e, l);
  const T f0 = d.has_pot ? phi[l] : T(0);
  if (d.hasx) {
    T v = vx[l];
    if (d.xwrap || i >= 1) {   // Eq. 53: density on the face = arithmetic mean
      const long long lm = d.id(d.xw(i - 1), j, k);
      const T il = d.invLX(j, k);
      const T wf = rdiv(T(2) * il, r0 + rho[lm]);
      T acc = wf * (p0 - pressure(d, rho, e, lm));
      if (d.has_pot) acc = rfma(f0 - phi[lm], il, acc);
      v = rfma(-dt, acc, vx[l]);
    }
    vxb[l] = v;
  }
  if (d.hasy) {
    T v = vy[l];
    if (j >= 1 && (!curv || ipok) && (!(sph && d.hasz) || k + 1 < d.TZ)) {
      const long long lm = l - d.pitch;
      const T il = d.invDY[j];
      const T wf = rdiv(T(2) * il, r0 + rho[lm]);
      T acc = wf * (p0 - pressure(d, rho, e, lm));
      if (d.has_pot) acc = rfma(f0 - phi[lm], il, acc);
      v = rfma(-dt, acc, vy[l]);
      if (curv) {   // Eq. 38: average the velocities, add the frame term, square (reading G27)
        const long long lp = d.id(ip, j, k);
        const T vphi = rfma(T(0.25), ((vx[l] + vx[lp]) + vx[lm]) + vx[lp - d.pitch], om * (d.ye[j] * d.Rxk[k]));
        T G = vphi * vphi;
        if (sph && d.hasz) {   // Eq. 36: + v_theta^2
          const T vth = T(0.25) * (((vz[l] + vz[l + d.plane]) + vz[lm]) + vz[lm + d.plane]);
          G = rfma(vth, vth, G);
        }
        v = rfma(dt, G * d.inv_ye[j], v);
      }
      if (d.shear) {   // Eq. 29: + 2 Omega_f v_x - 4 A Omega_f y on the Y face, v_x averaged as in Eq. 38 (G32)
        const long long lp = d.id(ip, j, k);
        const T vxa = T(0.25) * (((vx[l] + vx[lp]) + vx[lm]) + vx[lp - d.pitch]);
        v = rfma(dt, rfma(d.two_om, vxa, -(d.four_a_om * d.ye[j])), v);
      }
    }
    vyb[l] = v;
  }
  if (d.hasz) {
    T v = vz[l];
    if (k >= 1 && (!sph || ipok)) {
      const long long lm = l - d.plane;
      const T il = d.invDZ(j, k);
      const T wf = rdiv(T(2) * il, r0 + rho[lm]);
      T acc = wf * (p0 - pressure(d, rho, e, lm));
      if (d.has_pot) acc = rfma(f0 - phi[lm], il, acc);
      v = rfma(-dt, acc, vz[l]);
      if (sph) {   // Eq. 37: (v_phi^t)^2 cot(theta) / r on the theta face
        const long long lp = d.id(ip, j, k);
        const T vphi = rfma(T(0.25), ((vx[l] + vx[lp]) + vx[lm]) + vx[lp - d.plane], om * (d.yc[j] * d.sin_ze[k]));
        v = rfma(dt, ((vphi * vphi) * d.cot_ze[k]) * d.inv_yc[j], v);
      }
    }
    vzb[l] = v;
  }
}

template <typename T>
int launch_source_a(const Dev<T>& d, const State<T>& st, const T* phi, T* vxb, T* vyb, T* vzb, cudaStream_t s) {
  dim3 b(128), g((d.TX + 127) / 128, d.TY, d.TZ);
  k_source_a<T><<<g, b, 0, s>>>(d, st, phi, vxb, vyb, vzb);
  return 1;
}

// ---- 7b ---------------------------------------------------------------------------------------------
// q_d = C_q^2 rho (dv_d)^2 where dv_d < 0, else 0; evaluated on the fly for the cell and its lower
// neighbour in each direction (never stored).
template <typename T>
__device__ __forceinline__ T qvisc(const T cq2, const T rho, const T dv) {
  return dv < T(0) ? (cq2 * rho) * (dv * dv) : T(0);
}

template <typename T>
__global__ void __launch_bounds__(128) k_source_b(const Dev<T> d, const State<T> st, const T* __restrict__ vxb,
                                                  const T* __restrict__ vyb, const T* __restrict__ vzb,
                                                  T* __restrict__ vxc, T* __restrict__ vyc, T* __restrict__ vzc,
                                                  T* __restrict__ ec) {
  if (d.ctl->done) return;
  const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y, k = blockIdx.z;
  if (i >= d.TX) return;
  const T dt = (T)d.ctl->dt, cq2 = d.cvnr2;
  const long long l = d.id(i, j, k);
  const T* __restrict__ rho = st.rho;
  const T r0 = rho[l];
  T heat = T(0);
  if (d.hasx) {
    const T v0 = vxb[l];
    T dv = T(0), q = T(0);
    if (d.xwrap || i + 1 < d.TX) { dv = vxb[d.id(d.xw(i + 1), j, k)] - v0; q = qvisc(cq2, r0, dv); }
    T v = v0;
    if (d.xwrap || i >= 1) {
      const long long lm = d.id(d.xw(i - 1), j, k);
      const T rm = rho[lm];
      const T qm = qvisc(cq2, rm, v0 - vxb[lm]);   // q of the lower neighbour: its dv = v0 - vb[lm]
      const T wf = rdiv(T(2) * d.invLX(j, k), r0 + rm);
      v = rfma(-dt, wf * (q - qm), v0);
    }
    vxc[l] = v;
    heat = (q * dv) * d.invLX(j, k);
  }
  if (d.hasy) {
    const T v0 = vyb[l];
    T dv = T(0), q = T(0);
    if (j + 1 < d.TY) { dv = vyb[l + d.pitch] - v0; q = qvisc(cq2, r0, dv); }
    T v = v0;
    if (j >= 1) {
      const long long lm = l - d.pitch;
      const T rm = rho[lm];
      const T qm = qvisc(cq2, rm, v0 - vyb[lm]);
      const T wf = rdiv(T(2) * d.invDY[j], r0 + rm);
      v = rfma(-dt, wf * (q - qm), v0);
    }
    vyc[l] = v;
    heat = rfma(q * dv, d.invLY[j], heat);
  }
  if (d.hasz) {
    const T v0 = vzb[l];
    T dv = T(0), q = T(0);
    if (k + 1 < d.TZ) { dv = vzb[l + d.plane] - v0; q = qvisc(cq2, r0, dv); }
    T v = v0;
    if (k >= 1) {
      const long long lm = l - d.plane;
      const T rm = rho[lm];
      const T qm = qvisc(cq2, rm, v0 - vzb[lm]);
      const T wf = rdiv(T(2) * d.invDZ(j, k), r0 + rm);
      v = rfma(-dt, wf * (q - qm), v0);
    }
    vzc[l] = v;
    heat = rfma(q * dv, d.invLZ(j, k), heat);
  }
  if (d.eos == EOS_ADI) ec[l] = rfma(-dt, heat, st.e[l]);   // heating -q_d dv_d / Delta_d (G19)
}

template <typename T>
int launch_source_b(const Dev<T>& d, const State<T>& st, const T* vxb, const T* vyb, const T* vzb, T* vxc, T* vyc,
                    T* vzc, T* ec, cudaStream_t s) {
  dim3 b(128), g((d.TX + 127) / 128, d.TY, d.TZ);
  k_source_b<T><<<g, b, 0, s>>>(d, st, vxb, vyb, vzb, vxc, vyc, vzc, ec);
  return 1;
}

// ---- 7c ---------------------------------------------------------------------------------------------
template <typename T>
__global__ void __launch_bounds__(128) k_source_c(const Dev<T> d, const T* __restrict__ vxc, const T* __restrict__ vyc,
                                                  const T* __restrict__ vzc, const T* __restrict__ ec,
                                                  T* __restrict__ ed) {
  if (d.ctl->done) return;
  const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y, k = blockIdx.z;
  if (i >= d.TX) return;
  const T hd = (T(0.5) * (T)d.ctl->dt) * d.gm1;
  const long long l = d.id(i, j, k);
  T v = ec[l];
  const bool ok = (!d.hasx || d.xwrap || i + 1 < d.TX) && (!d.hasy || j + 1 < d.TY) && (!d.hasz || k + 1 < d.TZ);
  if (ok) {
    T tx = T(0), ty = T(0), tz = T(0);
    if (d.hasx) tx = (vxc[d.id(d.xw(i + 1), j, k)] - vxc[l]) * d.Sx(j, k);
    if (d.hasy) ty = rfma(vyc[l + d.pitch], d.Sy(j + 1, k), -(vyc[l] * d.Sy(j, k)));
    if (d.hasz) tz = rfma(vzc[l + d.plane], d.Sz(j, k + 1), -(vzc[l] * d.Sz(j, k)));
    const T D = d.invV(j, k) * ((tx + ty) + tz);
    const T a = hd * D;
    v = rdiv(ec[l] * (T(1) - a), T(1) + a);
  }
  ed[l] = v;
}

template <typename T>
int launch_source_c(const Dev<T>& d, const T* vxc, const T* vyc, const T* vzc, const T* ec, T* ed, cudaStream_t s) {
  dim3 b(128), g((d.TX + 127) / 128, d.TY, d.TZ);
  k_source_c<T><<<g, b, 0, s>>>(d, vxc, vyc, vzc, ec, ed);
  return 1;
}

// ---- 7b + 7c fused (adiabatic) ----------------------------------------------------------------------------
// e_d of a cell needs v_c on its six faces, and v_c on a face needs q on both sides of it, so per direction
// the thread forms q at m-1, m, m+1 from v_b at m-1 .. m+2 and v_c at m and m+1: one extra q and one extra
// division per direction against the two separate kernels, in exchange for never writing e_c and never
// re-reading v_c (9 reals per cell instead of 14).  Every expression is the one k_source_b / k_source_c
// evaluate for the same face, so the results are bit-identical to the two-kernel sequence.
template <typename T>
struct FaceBC { T vc0, vc1, qdv; };   // v_c on the lower and upper face of the cell, q dv of the cell

// one direction: vb[] = v_b at m-1, m, m+1, m+2; rr[] = rho at m-1, m, m+1; have* say which exist;
// il0 / il1 = inverse centre distance across the lower / upper face
template <typename T>
__device__ __forceinline__ FaceBC<T> face_bc(const T cq2, const T dt, const T vbm, const T vb0, const T vb1,
                                             const T vb2, const T rm, const T r0, const T r1, const bool has_m,
                                             const bool has_1, const bool has_2, const T il0, const T il1) {
  FaceBC<T> o;
  T dv = T(0), q = T(0);
  if (has_1) { dv = vb1 - vb0; q = qvisc(cq2, r0, dv); }
  o.vc0 = vb0;
  if (has_m) {
    const T qm = qvisc(cq2, rm, vb0 - vbm);
    const T wf = rdiv(T(2) * il0, r0 + rm);
    o.vc0 = rfma(-dt, wf * (q - qm), vb0);
  }
  o.vc1 = vb1;
  if (has_1) {   // the upper face: what k_source_b computes at the upper neighbour
    T q1 = T(0);
    if (has_2) q1 = qvisc(cq2, r1, vb2 - vb1);
    const T wf = rdiv(T(2) * il1, r1 + r0);
    o.vc1 = rfma(-dt, wf * (q1 - q), vb1);
  }
  o.qdv = q * dv;
  return o;
}

template <typename T>
__global__ void __launch_bounds__(128) k_source_bc(const Dev<T> d, const State<T> st, const T* __restrict__ vxb,
                                                   const T* __restrict__ vyb, const T* __restrict__ vzb,
                                                   T* __restrict__ vxc, T* __restrict__ vyc, T* __restrict__ vzc,
                                                   T* __restrict__ ed) {
  if (d.ctl->done) return;
  const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y, k = blockIdx.z;
  if (i >= d.TX) return;
  const T dt = (T)d.ctl->dt, cq2 = d.cvnr2;
  const long long l = d.id(i, j, k);
  const T* __restrict__ rho = st.rho;
  const T r0 = rho[l];
  T heat = T(0), tx = T(0), ty = T(0), tz = T(0);
  bool ok = true;
  if (d.hasx) {
    const bool w = d.xwrap != 0;
    const bool hm = w || i >= 1, h1 = w || i + 1 < d.TX, h2 = w || i + 2 < d.TX;
    const long long row = l - i;
    const long long lm = row + d.xw(i - 1), l1 = row + d.xw(i + 1), l2 = row + d.xw(i + 2);
    const T il = d.invLX(j, k);
    const FaceBC<T> f = face_bc<T>(cq2, dt, hm ? vxb[lm] : T(0), vxb[l], h1 ? vxb[l1] : T(0), h2 ? vxb[l2] : T(0),
                                   hm ? rho[lm] : T(0), r0, h1 ? rho[l1] : T(0), hm, h1, h2, il, il);
    vxc[l] = f.vc0;
    heat = f.qdv * il;
    ok = ok && h1;
    tx = (f.vc1 - f.vc0) * d.Sx(j, k);
  }
  if (d.hasy) {
    const bool hm = j >= 1, h1 = j + 1 < d.TY, h2 = j + 2 < d.TY;
    const long long p = d.pitch;
    const FaceBC<T> f = face_bc<T>(cq2, dt, hm ? vyb[l - p] : T(0), vyb[l], h1 ? vyb[l + p] : T(0),
                                   h2 ? vyb[l + 2 * p] : T(0), hm ? rho[l - p] : T(0), r0, h1 ? rho[l + p] : T(0), hm,
                                   h1, h2, d.invDY[j], h1 ? d.invDY[j + 1] : T(0));
    vyc[l] = f.vc0;
    heat = rfma(f.qdv, d.invLY[j], heat);
    ok = ok && h1;
    if (h1) ty = rfma(f.vc1, d.Sy(j + 1, k), -(f.vc0 * d.Sy(j, k)));
  }
  if (d.hasz) {
    const bool hm = k >= 1, h1 = k + 1 < d.TZ, h2 = k + 2 < d.TZ;
    const long long p = d.plane;
    const FaceBC<T> f = face_bc<T>(cq2, dt, hm ? vzb[l - p] : T(0), vzb[l], h1 ? vzb[l + p] : T(0),
                                   h2 ? vzb[l + 2 * p] : T(0), hm ? rho[l - p] : T(0), r0, h1 ? rho[l + p] : T(0), hm,
                                   h1, h2, d.invDZ(j, k), h1 ? d.invDZ(j, k + 1) : T(0));
    vzc[l] = f.vc0;
    heat = rfma(f.qdv, d.invLZ(j, k), heat);
    ok = ok && h1;
    if (h1) tz = rfma(f.vc1, d.Sz(j, k + 1), -(f.vc0 * d.Sz(j, k)));
  }
  const T ec = rfma(-dt, heat, st.e[l]);   // heating -q_d dv_d / Delta_d (G19)
  T v = ec;
  if (ok) {
    const T hd = (T(0.5) * dt) * d.gm1;
    const T D = d.invV(j, k) * ((tx + ty) + tz);
    const T a = hd * D;
    v = rdiv(ec * (T(1) - a), T(1) + a);
  }
  ed[l] = v;
}

template <typename T>
int launch_source_bc(const Dev<T>& d, const State<T>& st, const T* vxb, const T* vyb, const T* vzb, T* vxc, T* vyc,
                     T* vzc, T* ed, cudaStream_t s) {
  dim3 b(128), g((d.TX + 127) / 128, d.TY, d.TZ);
  k_source_bc<T><<<g, b, 0, s>>>(d, st, vxb, vyb, vzb, vxc, vyc, vzc, ed);
  return 1;
}

// ---- 7d: 2-D cylindrical (phi, r), wrapped X --------------------------------------------------------------
// Centring: diagonal stresses at cell centres, tau_phi_r at the cell corner with the lowest
// phi and r.  Density at the corner = mean of the four cells around it (reading G24).
template <typename T>
__global__ void __launch_bounds__(128) k_visc_tensor(const Dev<T> d, const T* __restrict__ rho, const T* __restrict__ vx,
                                                     const T* __restrict__ vy, T* __restrict__ tpp, T* __restrict__ trr,
                                                     T* __restrict__ tpr) {
  if (d.ctl->done) return;
  const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y, k = 0;
  if (i >= d.TX) return;
  const T nu = d.nu, two3 = T(2) / T(3);
  const long long l = d.id(i, j, k), lip = d.id(d.xw(i + 1), j, k), lim = d.id(d.xw(i - 1), j, k);
  const T il = d.invLX(j, k);
  T a = T(0), b = T(0), c = T(0);
  if (j + 1 < d.TY) {
    const long long ljp = l + d.pitch;
    const T div = d.invV(j, k) * ((vx[lip] - vx[l]) * d.Sx(j, k) + (vy[ljp] * d.Sy(j + 1, k) - vy[l] * d.Sy(j, k)));
    const T mrn = -(rho[l] * nu);
    a = mrn * (T(2) * ((vx[lip] - vx[l]) * il + (T(0.5) * (vy[l] + vy[ljp])) * d.inv_yc[j]) - two3 * div);
    b = mrn * (T(2) * ((vy[ljp] - vy[l]) * d.invLY[j]) - two3 * div);
  }
  if (j >= 1) {
    const long long ljm = l - d.pitch, limjm = lim - d.pitch;
    const T rhob = T(0.25) * (((rho[l] + rho[lim]) + rho[ljm]) + rho[limjm]);
    const T ilf = d.inv_ye[j] * d.invdx;   // 1/(r_f dphi)
    c = -(rhob * nu) * (((vx[l] - vx[ljm]) * d.invDY[j] - (T(0.5) * (vx[l] + vx[ljm])) * d.inv_ye[j])
                        + (vy[l] - vy[lim]) * ilf);
  }
  tpp[l] = a; trr[l] = b; tpr[l] = c;
}

template <typename T>
__global__ void __launch_bounds__(128) k_visc_force(const Dev<T> d, const T* __restrict__ rho, const T* __restrict__ vx,
                                                    const T* __restrict__ vy, const T* __restrict__ tpp,
                                                    const T* __restrict__ trr, const T* __restrict__ tpr,
                                                    T* __restrict__ vxd, T* __restrict__ vyd) {
  if (d.ctl->done) return;
  const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y, k = 0;
  if (i >= d.TX) return;
  const T dt = (T)d.ctl->dt;
  const long long l = d.id(i, j, k), lip = d.id(d.xw(i + 1), j, k), lim = d.id(d.xw(i - 1), j, k);
  T ox = vx[l], oy = vy[l];
  if (j >= 1 && j + 1 < d.TY) {
    const long long ljp = l + d.pitch, ljm = l - d.pitch;
    const T il = d.invLX(j, k), ilf = d.inv_ye[j] * d.invdx;
    const T y0 = d.ye[j], y1 = d.ye[j + 1];
    {   // B5, azimuthal: (1/r^2) d_r(r^2 tau_phi_r) + (1/r) d_phi tau_phi_phi
      const T a = (((y1 * y1) * tpr[ljp] - (y0 * y0) * tpr[l]) * (d.inv_yc[j] * d.inv_yc[j])) * d.invLY[j];
      const T b = (tpp[l] - tpp[lim]) * il;
      ox = vx[l] - dt * (rdiv(T(2), rho[l] + rho[lim]) * (a + b));
    }
    if (j >= 2) {   // B5, radial: (1/r) d_r(r tau_rr) + (1/r) d_phi tau_r_phi - tau_phi_phi / r
      const T a = ((d.yc[j] * trr[l] - d.yc[j - 1] * trr[ljm]) * d.inv_ye[j]) * d.invDY[j];
      const T b = (tpr[lip] - tpr[l]) * ilf;
      const T dd = (T(0.5) * (tpp[l] + tpp[ljm])) * d.inv_ye[j];
      oy = vy[l] - dt * (rdiv(T(2), rho[l] + rho[ljm]) * ((a + b) - dd));
    }
  }
  vxd[l] = ox; vyd[l] = oy;
}

template <typename T>
int launch_source_d(const Dev<T>& d, const T* rho, const T* vxc, const T* vyc, T* tpp, T* trr, T* tpr, T* vxd, T* vyd,
                    cudaStream_t s) {
  dim3 b(128), g((d.TX + 127) / 128, d.TY, 1);
  k_visc_tensor<T><<<g, b, 0, s>>>(d, rho, vxc, vyc, tpp, trr, tpr);
  k_visc_force<T><<<g, b, 0, s>>>(d, rho, vxc, vyc, tpp, trr, tpr, vxd, vyd);
  return 2;
}

#define INST(T)                                                                                                      \
  template int launch_source_bc<T>(const Dev<T>&, const State<T>&, const T*, const T*, const T*, T*, T*, T*, T*,     \
                                   cudaStream_t);                                                                    \
  template int launch_source_a<T>(const Dev<T>&, const State<T>&, const T*, T*, T*, T*, cudaStream_t);               \
  template int launch_source_b<T>(const Dev<T>&, const State<T>&, const T*, const T*, const T*, T*, T*, T*, T*,      \
                                  cudaStream_t);                                                                     \
  template int launch_source_c<T>(const Dev<T>&, const T*, const T*, const T*, const T*, T*, cudaStream_t);          \
  template int launch_source_d<T>(const Dev<T>&, const T*, const T*, const T*, T*, T*, T*, T*, T*, cudaStream_t);
INST(double)
INST(float)
#undef INST

}  // namespace fg
