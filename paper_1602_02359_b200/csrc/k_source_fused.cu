// k_source_fused.cu -- the whole operator-split source step (Fig. 2 cells 7a + 7b + 7c) as ONE
// pass over the mesh for 3-D meshes with a wrapped X axis: the state (rho, e, v [, Phi]) is read once and the
// source-updated (e, v) written once, 72 B per cell (adiabatic) instead of the 136 B of k_source_a +
// k_source_bc.  The intermediates v_b (after 7a) and q (7b) are never stored.
//
// Only ACTIVE cells are produced (the ghost fill of cell 9 overwrites every ghost of e and v before anything
// reads them), so every stencil below stays inside the 3 ghost layers and no bounds test is needed.
//
// Work decomposition (no shared memory, no barriers):
//   X : a warp owns 64 consecutive cells of a row, two per lane (16-byte vector accesses); v_b, q and v_c of
//       the X faces cross lanes by shuffle; lanes 0 and 31 are recomputed halo (60 cells stored per warp).
//   Z : the thread marches along Z; v_b, q, v_c of the Z faces live in registers.  Plane m = n - 2 is finished
//       when plane n has been read.  The thread's own row (rho, e, v [, Phi]) is fetched SF_RD planes ahead with
//       16-byte cp.async into a ring of SF_RS slots private to the thread (no barrier: a thread reads only what
//       it copied itself); the ring also keeps planes n-1 and n-2, so nothing of the state is carried in
//       registers.
//   Y : v_b of the Y faces of rows j-1 .. j+2 is recomputed from the neighbour rows' state (served by L1/L2:
//       the four warps of a block are four consecutive rows); one division per recomputed face.
// Every expression is the one k_source_a / k_source_b / k_source_c evaluate for the same face or cell, in the
// same order, so the result is bit-identical to the three-kernel sequence (tests: whole-step parity).
#include "kernels.h"

namespace fg {

template <typename T> struct SPair;
template <> struct SPair<double> { using type = double2; };
template <> struct SPair<float> { using type = float2; };

template <typename T> struct V2 { T a, b; };

template <typename T>
__device__ __forceinline__ V2<T> ldv(const T* __restrict__ p) {
  const typename SPair<T>::type v = *reinterpret_cast<const typename SPair<T>::type*>(p);
  V2<T> o; o.a = v.x; o.b = v.y; return o;
}
template <typename T>
__device__ __forceinline__ void stv(T* __restrict__ p, const T a, const T b) {
  typename SPair<T>::type v; v.x = a; v.y = b;
  *reinterpret_cast<typename SPair<T>::type*>(p) = v;
}
template <typename T> __device__ __forceinline__ T s_up1(T v) { return __shfl_up_sync(0xffffffffu, v, 1); }
template <typename T> __device__ __forceinline__ T s_dn1(T v) { return __shfl_down_sync(0xffffffffu, v, 1); }

template <typename T>
__device__ __forceinline__ T qv(const T cq2, const T rho, const T dv) {   // readings G8, G19
  return dv < T(0) ? (cq2 * rho) * (dv * dv) : T(0);
}
template <typename T, bool ADI>
__device__ __forceinline__ T eos_p(const T gm1, const T e, const T rho) {   // Eq. 7 | Eq. 6
  return ADI ? gm1 * e : (e * e) * rho;
}

constexpr int SFW = 4;        // warps (consecutive rows) per block
constexpr int SFIN = 60;      // cells stored per warp
// One plane in flight: the ring goes through L1 (cp.async.ca) and the neighbour rows are served by L1 as well, so a short
// ring that leaves more of the 256 KB to L1 wins (three planes in flight: 2.89 ms at 512^3, one: 2.67 ms; profiles/r02a).
constexpr int SF_RD = 1;             // planes in flight
constexpr int SF_RS = SF_RD + 3;     // ring slots: planes n-2 .. n+SF_RD

__device__ __forceinline__ void sf_cp_pair(unsigned dst, const double* src) {   // one pair of cells
  asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void sf_cp_pair(unsigned dst, const float* src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void sf_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void sf_prefetch_l1(const void* p) { asm volatile("prefetch.global.L1 [%0];" ::"l"(p)); }
template <int N> __device__ __forceinline__ void sf_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

template <typename T, int GEO, bool ADI, bool POT, bool RING>
__global__ void __launch_bounds__(32 * SFW, 3) k_source_fused(const Dev<T> d, const State<T> st, const T* __restrict__ phi,
                                                           const State<T> out, const int CH, const int ext) {
  constexpr bool CURV = GEO == GEO_CYL || GEO == GEO_SPH, SPH = GEO == GEO_SPH;
  constexpr bool SHEAR = GEO == GEO_SHEAR;   // shearing sheet: Cartesian metric + Eq. 29 on the Y faces (reading G32)
  constexpr bool VXR = CURV || SHEAR;        // the Y faces need v_x of the neighbour rows
  constexpr int NV = ADI ? 4 : 3;   // Y faces whose v_b is needed: rows j-1 .. j-2+NV (7c needs v_c on the upper face too)
  if (d.ctl->done) return;
  const int lane = threadIdx.x;
  // ext = 1 (viscosity follows): one ghost layer more in Y and Z, where 7d reads v_c (its stencil still fits in
  // the three ghost layers: rows j-2 .. j+2, planes m-2 .. m+1)
  const int j = d.ngy - ext + blockIdx.y * SFW + threadIdx.y;
  if (j >= d.ngy + d.ny + ext) return;   // whole warps leave together
  const int m0 = d.ngz - ext + blockIdx.z * CH;
  const int mend = d.ngz + d.nz + ext;
  const int m1 = (m0 + CH < mend) ? m0 + CH : mend;   // planes this thread writes: [m0, m1)
  const int iu = blockIdx.x * SFIN - 2 + 2 * lane;   // un-wrapped index of the lane's first cell (even)
  int i = iu % d.nx; if (i < 0) i += d.nx;
  const bool store = lane >= 1 && lane <= 30 && iu < d.nx;
  const T dt = (T)d.ctl->dt, cq2 = d.cvnr2, gm1 = d.gm1, om = d.omega;
  const long long P = d.plane, R = d.pitch;
  const long long base = d.id(i, j, 0);
  const T* __restrict__ rho = st.rho;
  const T* __restrict__ en = st.e;
  const T* __restrict__ vx = st.vx;
  const T* __restrict__ vy = st.vy;
  const T* __restrict__ vz = st.vz;

  // per-row geometry (Tab. 5 factors of this row and of the rows whose Y face is recomputed)
  T ilY[NV], yeR[NV], iyeR[NV];
#pragma unroll
  for (int t = 0; t < NV; ++t) {
    ilY[t] = d.invDY[j - 1 + t];
    yeR[t] = VXR ? d.ye[j - 1 + t] : T(0);
    iyeR[t] = CURV ? d.inv_ye[j - 1 + t] : T(0);
  }
  const T invLXj = d.invLXj[j], invRzj = d.invRzj[j], invLYj = d.invLY[j];
  const T sxj = d.sxj[j], syj0 = d.syj[j], syj1 = d.syj[j + 1], szj = d.szj[j], invVj = d.invVj[j];
  const T ycj = d.yc[j], iycj = d.inv_yc[j];

  // ring of the thread's own row: slot s, array a at ((s * NAO + a) * 128 + tid) pairs; arrays: rho e vz vx vy [Phi]
  constexpr int NAO = POT ? 6 : 5;
  using P2 = typename SPair<T>::type;
  extern __shared__ __align__(16) unsigned char sf_smem[];
  const int tid = threadIdx.y * 32 + lane;
  P2* const ring = reinterpret_cast<P2*>(sf_smem) + tid;
  const unsigned ring_s = (unsigned)__cvta_generic_to_shared(ring);
  const int nlast = m1 + 1;
  auto fetch = [&](const int n) {
    if (!RING) return;
    if (n <= nlast) {
      const long long l = base + (long long)n * P;
      const unsigned dst = ring_s + (unsigned)(((n % SF_RS) * NAO) * 128 * sizeof(P2));
      sf_cp_pair(dst, rho + l);
      sf_cp_pair(dst + (unsigned)(1 * 128 * sizeof(P2)), en + l);
      sf_cp_pair(dst + (unsigned)(2 * 128 * sizeof(P2)), vz + l);
      sf_cp_pair(dst + (unsigned)(3 * 128 * sizeof(P2)), vx + l);
      sf_cp_pair(dst + (unsigned)(4 * 128 * sizeof(P2)), vy + l);
      if (POT) sf_cp_pair(dst + (unsigned)(5 * 128 * sizeof(P2)), phi + l);
    }
    sf_commit();   // one group per plane, empty past the end
  };
  auto own = [&](const int n, const int a) -> V2<T> {
    if (!RING) {   // curvilinear meshes read many neighbour rows: they keep the whole L1 instead of a ring
      const T* const arr = a == 0 ? rho : a == 1 ? en : a == 2 ? vz : a == 3 ? vx : a == 4 ? vy : phi;
      return ldv(arr + base + (long long)n * P);
    }
    const P2 v = ring[((n % SF_RS) * NAO + a) * 128];
    V2<T> o; o.a = v.x; o.b = v.y; return o;
  };
#pragma unroll
  for (int q = 0; q < SF_RD; ++q) fetch(m0 - 2 + q);

  // carried along Z (index 1 = plane n-1, 2 = plane n-2): only what was computed, the state is in the ring
  const V2<T> zero = {T(0), T(0)};
  V2<T> vbz1 = zero, wfz1 = zero, qz2 = zero, hz2 = zero, vcz2 = zero;

#pragma unroll 1
  for (int n = m0 - 2; n <= m1 + 1; ++n) {
    fetch(n + SF_RD);
    if (n + 1 >= m0 + 2 && n + 1 <= nlast) {   // next plane's neighbour rows: into L1 while this plane is reduced
      const long long lq = base + (long long)(n - 1) * P;
#pragma unroll
      for (int t = 0; t <= NV; ++t) {
        if (t == 2) continue;
        const long long lr = lq + (long long)(t - 2) * R;
        sf_prefetch_l1(rho + lr);
        sf_prefetch_l1(en + lr);
        if (POT) sf_prefetch_l1(phi + lr);
        if (t >= 1) sf_prefetch_l1(vy + lr);
        if (VXR) sf_prefetch_l1(vx + lr);
        if (SPH) { sf_prefetch_l1(vz + lr); sf_prefetch_l1(vz + lr + P); }
      }
    }
    if (RING) sf_wait<SF_RD>();   // plane n has landed
    // ---- leading plane n: v_b, q, v_c of the Z faces -------------------------------------------------------
    const bool warm = n > m0 - 2;   // plane n-1 is in the ring
    const V2<T> rn = own(n, 0), en_ = own(n, 1), vzn = own(n, 2);
    const V2<T> r1 = warm ? own(n - 1, 0) : rn, e1 = warm ? own(n - 1, 1) : en_;
    V2<T> fn = zero, f1 = zero, vxn = zero, vx1 = zero;
    if (POT) { fn = own(n, 5); f1 = warm ? own(n - 1, 5) : fn; }
    if (SPH) { vxn = own(n, 3); vx1 = warm ? own(n - 1, 3) : vxn; }
    V2<T> p1;
    p1.a = eos_p<T, ADI>(gm1, e1.a, r1.a);
    p1.b = eos_p<T, ADI>(gm1, e1.b, r1.b);
    V2<T> pn;
    pn.a = eos_p<T, ADI>(gm1, en_.a, rn.a);
    pn.b = eos_p<T, ADI>(gm1, en_.b, rn.b);
    const T ilz = d.invdzc[n] * invRzj;
    V2<T> vbz, wfz, qz1, hz1, vcz1;
    T geo_z = T(0), frame_z = T(0);
    if (SPH) { geo_z = d.cot_ze[n]; frame_z = om * (ycj * d.sin_ze[n]); }
    const T vxn_r = SPH ? s_dn1(vxn.a) : T(0), vx1_r = SPH ? s_dn1(vx1.a) : T(0);
#pragma unroll
    for (int c = 0; c < 2; ++c) {
      const T rN = c ? rn.b : rn.a, rL = c ? r1.b : r1.a, pN = c ? pn.b : pn.a, pL = c ? p1.b : p1.a;
      const T w = rdiv(T(2) * ilz, rN + rL);
      T acc = w * (pN - pL);
      if (POT) acc = rfma((c ? fn.b : fn.a) - (c ? f1.b : f1.a), ilz, acc);
      T v = rfma(-dt, acc, c ? vzn.b : vzn.a);
      if (SPH) {   // Eq. 37: (v_phi^t)^2 cot(theta) / r on the theta face (reading G27)
        const T x00 = c ? vxn.b : vxn.a, x10 = c ? vxn_r : vxn.b, x01 = c ? vx1.b : vx1.a, x11 = c ? vx1_r : vx1.b;
        const T vphi = rfma(T(0.25), ((x00 + x10) + x01) + x11, frame_z);
        v = rfma(dt, ((vphi * vphi) * geo_z) * iycj, v);
      }
      const T vprev = c ? vbz1.b : vbz1.a;
      const T dv = v - vprev;
      const T q = qv(cq2, rL, dv);                                      // q of plane n-1
      const T vc = rfma(-dt, (c ? wfz1.b : wfz1.a) * (q - (c ? qz2.b : qz2.a)), vprev);   // v_c, lower Z face of plane n-1
      if (c) { vbz.b = v; wfz.b = w; qz1.b = q; hz1.b = q * dv; vcz1.b = vc; }
      else { vbz.a = v; wfz.a = w; qz1.a = q; hz1.a = q * dv; vcz1.a = vc; }
    }

    if (n >= m0 + 2) {
      // ---- plane m = n - 2: X and Y faces, then the cell ---------------------------------------------------
      const int m = n - 2;
      const long long lm = base + (long long)m * P;
      const V2<T> r2 = own(m, 0), e2 = own(m, 1), f2 = POT ? own(m, 5) : zero;
      V2<T> p2;
      p2.a = eos_p<T, ADI>(gm1, e2.a, r2.a);
      p2.b = eos_p<T, ADI>(gm1, e2.b, r2.b);
      V2<T> rr[NV + 1], pp[NV + 1], ff[NV + 1], vyr[NV + 1], vxr[NV + 1], vz0[NV + 1], vz1[NV + 1];
#pragma unroll
      for (int t = 0; t <= NV; ++t) {
        const long long lr = lm + (long long)(t - 2) * R;
        if (t == 2) { rr[t] = r2; pp[t] = p2; ff[t] = f2; }   // own row: from the ring
        else {
          rr[t] = ldv(rho + lr);
          const V2<T> ee = ldv(en + lr);
          pp[t].a = eos_p<T, ADI>(gm1, ee.a, rr[t].a);
          pp[t].b = eos_p<T, ADI>(gm1, ee.b, rr[t].b);
          ff[t] = POT ? ldv(phi + lr) : zero;
        }
        vyr[t] = t == 2 ? own(m, 4) : (t >= 1 ? ldv(vy + lr) : zero);
        vxr[t] = t == 2 ? own(m, 3) : (VXR ? ldv(vx + lr) : zero);
        vz0[t] = SPH ? (t == 2 ? own(m, 2) : ldv(vz + lr)) : zero;
        vz1[t] = SPH ? (t == 2 ? own(m + 1, 2) : ldv(vz + lr + P)) : zero;
      }
      const T il = invLXj * d.invRxk[m];
      // ---- X faces ----
      V2<T> vcx, hx, tx;
      {
        const T rL = s_up1(r2.b), pL = s_up1(p2.b), fL = POT ? s_up1(f2.b) : T(0);
        const T wA = rdiv(T(2) * il, r2.a + rL), wB = rdiv(T(2) * il, r2.b + r2.a);
        T accA = wA * (p2.a - pL), accB = wB * (p2.b - p2.a);
        if (POT) { accA = rfma(f2.a - fL, il, accA); accB = rfma(f2.b - f2.a, il, accB); }
        const T vbA = rfma(-dt, accA, vxr[2].a), vbB = rfma(-dt, accB, vxr[2].b);
        const T vbR = s_dn1(vbA);
        const T dvA = vbB - vbA, dvB = vbR - vbB;
        const T qA = qv(cq2, r2.a, dvA), qB = qv(cq2, r2.b, dvB);
        const T qL = s_up1(qB);
        vcx.a = rfma(-dt, wA * (qA - qL), vbA);
        vcx.b = rfma(-dt, wB * (qB - qA), vbB);
        const T vcR = s_dn1(vcx.a);
        hx.a = (qA * dvA) * il; hx.b = (qB * dvB) * il;
        const T Sx = sxj * d.sxk[m];
        tx.a = (vcx.b - vcx.a) * Sx; tx.b = (vcR - vcx.b) * Sx;
      }
      // ---- Y faces ----
      V2<T> vcy, hy = zero, ty = zero;
      {
        T vxn_t[NV + 1];   // vx of the right neighbour's first cell, per row (curvature terms)
#pragma unroll
        for (int t = 0; t <= NV; ++t) vxn_t[t] = VXR ? s_dn1(vxr[t].a) : T(0);
        const T Rxk = CURV ? d.Rxk[m] : T(0);
        const T Sy0 = syj0 * d.syk[m], Sy1 = syj1 * d.syk[m];
#pragma unroll
        for (int c = 0; c < 2; ++c) {
          T vby[NV + 1], wfy[NV + 1];
#pragma unroll
          for (int t = 1; t <= NV; ++t) {
            const T rT = c ? rr[t].b : rr[t].a, rB = c ? rr[t - 1].b : rr[t - 1].a;
            const T ily = ilY[t - 1];
            wfy[t] = rdiv(T(2) * ily, rT + rB);
            T acc = wfy[t] * ((c ? pp[t].b : pp[t].a) - (c ? pp[t - 1].b : pp[t - 1].a));
            if (POT) acc = rfma((c ? ff[t].b : ff[t].a) - (c ? ff[t - 1].b : ff[t - 1].a), ily, acc);
            T v = rfma(-dt, acc, c ? vyr[t].b : vyr[t].a);
            if (CURV) {   // Eq. 38: average the velocities, add the frame term, square (reading G27)
              const T x00 = c ? vxr[t].b : vxr[t].a, x10 = c ? vxn_t[t] : vxr[t].b;
              const T x01 = c ? vxr[t - 1].b : vxr[t - 1].a, x11 = c ? vxn_t[t - 1] : vxr[t - 1].b;
              const T vphi = rfma(T(0.25), ((x00 + x10) + x01) + x11, om * (yeR[t - 1] * Rxk));
              T G = vphi * vphi;
              if (SPH) {   // Eq. 36: + v_theta^2
                const T vth = T(0.25) * ((((c ? vz0[t].b : vz0[t].a) + (c ? vz1[t].b : vz1[t].a)) +
                                          (c ? vz0[t - 1].b : vz0[t - 1].a)) + (c ? vz1[t - 1].b : vz1[t - 1].a));
                G = rfma(vth, vth, G);
              }
              v = rfma(dt, G * iyeR[t - 1], v);
            }
            if (SHEAR) {   // Eq. 29: + 2 Omega_f v_x - 4 A Omega_f y, v_x averaged as in Eq. 38
              const T x00 = c ? vxr[t].b : vxr[t].a, x10 = c ? vxn_t[t] : vxr[t].b;
              const T x01 = c ? vxr[t - 1].b : vxr[t - 1].a, x11 = c ? vxn_t[t - 1] : vxr[t - 1].b;
              const T vxa = T(0.25) * (((x00 + x10) + x01) + x11);
              v = rfma(dt, rfma(d.two_om, vxa, -(d.four_a_om * yeR[t - 1])), v);
            }
            vby[t] = v;
          }
          T qy[NV];
#pragma unroll
          for (int t = 1; t < NV; ++t) qy[t] = qv(cq2, c ? rr[t].b : rr[t].a, vby[t + 1] - vby[t]);
          const T vc0 = rfma(-dt, wfy[2] * (qy[2] - qy[1]), vby[2]);
          if (c) vcy.b = vc0; else vcy.a = vc0;
          if (ADI) {
            const T vc1 = rfma(-dt, wfy[3] * (qy[NV - 1] - qy[2]), vby[3]);
            const T h = qy[2] * (vby[3] - vby[2]);   // q dv of the cell; scaled by 1/LY in the heating chain below
            const T tt = rfma(vc1, Sy1, -(vc0 * Sy0));
            if (c) { hy.b = h; ty.b = tt; } else { hy.a = h; ty.a = tt; }
          }
        }
      }
      // ---- the cell: 7b heating, 7c compression (readings G8, G19) ----
      st2_if(out.vx + lm, vcx.a, vcx.b, store);
      st2_if(out.vy + lm, vcy.a, vcy.b, store);
      st2_if(out.vz + lm, vcz2.a, vcz2.b, store);
      if (ADI) {
        const T ilZ = d.invdz[m] * invRzj;
        const T Sz0 = szj * d.szk[m], Sz1 = szj * d.szk[m + 1];
        const T iV = invVj * d.inv_syk[m];
        const T hd = (T(0.5) * dt) * gm1;
        T ed[2];
#pragma unroll
        for (int c = 0; c < 2; ++c) {
          T heat = c ? hx.b : hx.a;
          heat = rfma(c ? hy.b : hy.a, invLYj, heat);
          heat = rfma(c ? hz2.b : hz2.a, ilZ, heat);
          const T ec = rfma(-dt, heat, c ? e2.b : e2.a);
          const T tz = rfma(c ? vcz1.b : vcz1.a, Sz1, -((c ? vcz2.b : vcz2.a) * Sz0));
          const T D = iV * (((c ? tx.b : tx.a) + (c ? ty.b : ty.a)) + tz);
          const T a = hd * D;
          ed[c] = rdiv(ec * (T(1) - a), T(1) + a);
        }
        st2_if(out.e + lm, ed[0], ed[1], store);
      }
    }
    // ---- shift the Z window ----
    vbz1 = vbz; wfz1 = wfz; qz2 = qz1; hz2 = hz1; vcz2 = vcz1;
  }
  if (RING) sf_wait<0>();
}

template <typename T>
bool source_fused_ok(const Dev<T>& d) {
  return d.hasx && d.hasy && d.hasz && d.xwrap && d.nx % 2 == 0;   // with viscosity: followed by k_visc3d_fused
}

template <typename T, int GEO, bool ADI>
static int launch_sf(const Dev<T>& d, const State<T>& st, const T* phi, const State<T>& out, cudaStream_t s) {
  // chunk the march so that the grid fills the machine a few times over; each chunk re-reads 4 planes
  const int ext = d.visc ? 1 : 0;   // 7d reads v_c one ghost layer out in Y and Z
  const int nyo = d.ny + 2 * ext, nzo = d.nz + 2 * ext;
  const int ntile = (d.nx + SFIN - 1) / SFIN, nrow = (nyo + SFW - 1) / SFW;
  constexpr bool RING = GEO == GEO_CART || GEO == GEO_SHEAR;
  const size_t pair = 2 * sizeof(T);
  dim3 b(32, SFW);
  // chunks of the Z march: equal blocks run in rounds of the resident slots; each chunk re-reads 4 planes
  auto go = [&](auto kernel, const int sm) {
    static int slots = 0;   // per instantiation
    if (!slots) {
      if (RING) cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, sm);
      slots = resident_slots(kernel, 32 * SFW, (size_t)sm);
    }
    const int CH = pick_chunk_len((long long)ntile * nrow, nzo, 4, slots, 16);
    dim3 g(ntile, nrow, (nzo + CH - 1) / CH);
    kernel<<<g, b, sm, s>>>(d, st, phi, out, CH, ext);
  };
  if (d.has_pot) go(k_source_fused<T, GEO, ADI, true, RING>, RING ? (int)(SF_RS * 6 * 128 * pair) : 0);
  else go(k_source_fused<T, GEO, ADI, false, RING>, RING ? (int)(SF_RS * 5 * 128 * pair) : 0);
  return 1;
}

// cells 7a-7c in one pass: st -> out.{e (adiabatic), vx, vy, vz}; out.rho is not touched.  out must not alias st.
template <typename T>
int launch_source_fused(const Dev<T>& d, const State<T>& st, const T* phi, const State<T>& out, cudaStream_t s) {
  const bool adi = d.eos == EOS_ADI;
  if (d.shear) return adi ? launch_sf<T, GEO_SHEAR, true>(d, st, phi, out, s) : launch_sf<T, GEO_SHEAR, false>(d, st, phi, out, s);
  switch (d.geometry) {
    case GEO_CART: return adi ? launch_sf<T, GEO_CART, true>(d, st, phi, out, s) : launch_sf<T, GEO_CART, false>(d, st, phi, out, s);
    case GEO_CYL: return adi ? launch_sf<T, GEO_CYL, true>(d, st, phi, out, s) : launch_sf<T, GEO_CYL, false>(d, st, phi, out, s);
    default: return adi ? launch_sf<T, GEO_SPH, true>(d, st, phi, out, s) : launch_sf<T, GEO_SPH, false>(d, st, phi, out, s);
  }
}

#define INST(T)                                                                                              \
  template bool source_fused_ok<T>(const Dev<T>&);                                                           \
  template int launch_source_fused<T>(const Dev<T>&, const State<T>&, const T*, const State<T>&, cudaStream_t);
INST(double)
INST(float)
#undef INST

}  // namespace fg
