// k_transport.cu -- the transport step, box 12 of Fig. 2:
//   12a left/right momenta with the quantities of Tab. 2 (Eqs. 49-50; Tab. 2)
//   12b van Leer slopes and upwind star values at half time step (Eq. 48)
//   12c conservative update per direction (Eqs. 41-43, 45-47 P:292-326) with consistent transport:
//       q = Q/rho is reconstructed, the flux of Q is the mass flux times q*
//   12d new velocities (Eq. 51 P:355 + Tab. 2 inverted, reading G28)
//
// One sweep = ONE kernel: divide-by-rho, slope, star value, flux and update of rho and of every
// transported quantity are fused, so each field is read once and written once per direction
// (the paper runs ~4 kernels per field per direction).  No shared memory, no barriers:
//   X sweep  : one lane per cell, a warp owns 32 consecutive cells of a row (2 halo cells per side,
//              recomputed); neighbours' values, slopes and fluxes travel by warp shuffles.  On the
//              first pass the momenta are formed from the state in registers (12a fused).
//   Y/Z sweep: one thread per (i, line) marches along the sweep axis with a three-cell register
//              window; threads of a warp sit side by side along X, so every load and store is a
//              coalesced row segment.  The next row is loaded while the current one is reduced.
#include "kernels.h"

namespace fg {

// van Leer slope per unit length; zero unless both one-sided differences have the same sign (reading G4)
template <typename T>
__device__ __forceinline__ T vl_slope(const T fm, const T f0, const T fp, const T invd0, const T invdp) {
  const T dm = (f0 - fm) * invd0;
  const T dp = (fp - f0) * invdp;
  const T pr = dm * dp;
  const bool flat = pr <= T(0);
  const T den = flat ? T(1) : dm + dp;   // keeps the division on its fast path when the slope is dropped
  const T a = (T(2) * pr) / den;
  return flat ? T(0) : a;
}

template <typename T> __device__ __forceinline__ T shfl_up1(T v) { return __shfl_up_sync(0xffffffffu, v, 1); }
template <typename T> __device__ __forceinline__ T shfl_dn1(T v) { return __shfl_down_sync(0xffffffffu, v, 1); }

// ---- 12a alone: only when X is absent, so that the first sweep (Y or Z) can read a stored set ----------
template <typename T>
__global__ void __launch_bounds__(128) k_momenta(const Dev<T> d, const State<T> st, const QSet<T> S) {
  if (d.ctl->done) return;
  const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y, k = blockIdx.z;
  if (i >= d.TX) return;
  const long long l = d.id(i, j, k);
  const T r0 = st.rho[l], rz = d.Rzj[j];
  if (d.hasy) {
    const T v = st.vy[l];
    const T vp = j + 1 < d.TY ? st.vy[l + d.pitch] : v;
    S.q[3][l] = r0 * v;
    S.q[4][l] = r0 * vp;
  }
  if (d.hasz) {
    const T v = st.vz[l];
    const T vp = k + 1 < d.TZ ? st.vz[l + d.plane] : v;
    S.q[5][l] = r0 * (rz * v);
    S.q[6][l] = r0 * (rz * vp);
  }
}

template <typename T>
int launch_momenta(const Dev<T>& d, const State<T>& st, const QSet<T>& S, cudaStream_t s) {
  dim3 b(128), g((d.TX + 127) / 128, d.TY, d.TZ);
  k_momenta<T><<<g, b, 0, s>>>(d, st, S);
  return 1;
}

// ---- X sweep ------------------------------------------------------------------------------------------
constexpr int XW = 8;         // warps (rows) per block
constexpr int XIN = 28;       // interior cells per warp

template <typename T, int NQ, bool FIRST>
__global__ void __launch_bounds__(32 * XW) k_sweep_x(const Dev<T> d, const SweepArgs<T> A) {
  if (d.ctl->done) return;
  const int lane = threadIdx.x;
  const int j = blockIdx.y * XW + threadIdx.y, k = blockIdx.z;
  if (j >= d.TY) return;   // whole warps leave together
  const bool wrap = d.xwrap != 0;
  const int iu = blockIdx.x * XIN - 2 + lane;   // un-wrapped cell index
  int i = iu;
  if (wrap) { i %= d.nx; if (i < 0) i += d.nx; }
  const bool valid = i >= 0 && i < d.TX;
  const bool inner = valid && lane >= 2 && lane < 30 && iu < d.TX;
  const bool upd = inner && (wrap || (i >= 2 && i < d.TX - 2));

  const T dt = (T)d.ctl->dt;
  const T len = d.LX(j, k), invd = d.invLX(j, k), Sm = d.Sx(j, k), dtiv = dt * d.invV(j, k);
  const long long l = valid ? d.id(i, j, k) : d.id(0, j, k);

  T Q[NQ], r0 = T(1), w = T(0);
  if (valid) {
    r0 = A.srho[l];
    w = A.st.vx[l];
  }
  if (FIRST) {
    // momenta of Tab. 2 from the state (12a)
    T mom[7] = {T(0), T(0), T(0), T(0), T(0), T(0), T(0)};
    T wp = shfl_dn1(w);
    if (valid) {
      if (lane == 31) wp = (d.xwrap || i + 1 < d.TX) ? A.st.vx[d.id(d.xw(i + 1), j, k)] : w;
      else if (!d.xwrap && i + 1 >= d.TX) wp = w;
      const T rx = d.Rx(j, k), rx2om = (rx * rx) * d.om_eff, rz = d.Rzj[j];
      if (d.eos == EOS_ADI) mom[0] = A.st.e[l];
      mom[1] = r0 * (rx * w + rx2om);
      mom[2] = r0 * (rx * wp + rx2om);
      if (d.hasy) {
        const T v = A.st.vy[l];
        const T vp = j + 1 < d.TY ? A.st.vy[l + d.pitch] : v;
        mom[3] = r0 * v;
        mom[4] = r0 * vp;
      }
      if (d.hasz) {
        const T v = A.st.vz[l];
        const T vp = k + 1 < d.TZ ? A.st.vz[l + d.plane] : v;
        mom[5] = r0 * (rz * v);
        mom[6] = r0 * (rz * vp);
      }
    }
#pragma unroll
    for (int q = 0; q < NQ; ++q) {
      const int sl = A.slot[q];
      T v = mom[0];
#pragma unroll
      for (int s = 1; s < 7; ++s) v = (sl == s) ? mom[s] : v;
      Q[q] = v;
    }
  } else {
#pragma unroll
    for (int q = 0; q < NQ; ++q) Q[q] = valid ? A.sq[q][l] : T(0);
  }
  if (A.v0) w = w - A.v0[d.rid(j, k)];   // residual velocity under orbital advection
  const bool up = w >= T(0);              // reading G3: ties go to the first branch
  const T wdt = w * dt;
  const T hup = (len - wdt) * T(0.5), hdn = (len + wdt) * T(0.5);   // Eq. 48
  const T ir = T(1) / r0;

  // density: its mass flux F = w rho* S multiplies every other star value
  T Fr;
  {
    const T fm = shfl_up1(r0), fp = shfl_dn1(r0);
    const T a = vl_slope(fm, r0, fp, invd, invd);
    const T am = shfl_up1(a);
    const T rs = up ? fm + am * hup : r0 - a * hdn;
    Fr = (w * rs) * Sm;
    const T Fp = shfl_dn1(Fr);
    if (inner) A.drho[l] = upd ? r0 - dtiv * (Fp - Fr) : r0;
  }
#pragma unroll
  for (int q = 0; q < NQ; ++q) {
    const T f = Q[q] * ir;
    const T fm = shfl_up1(f), fp = shfl_dn1(f);
    const T a = vl_slope(fm, f, fp, invd, invd);
    const T am = shfl_up1(a);
    const T fs = up ? fm + am * hup : f - a * hdn;
    const T F = Fr * fs;
    const T Fp = shfl_dn1(F);
    if (inner) A.dq[q][l] = upd ? Q[q] - dtiv * (Fp - F) : Q[q];
  }
}

// ---- Y / Z sweep: register marching -----------------------------------------------------------------------
constexpr int MTHREADS = 128;

template <typename T, int DIR, int NQ>
__global__ void __launch_bounds__(MTHREADS) k_sweep_march(const Dev<T> d, const SweepArgs<T> A, const int CH) {
  if (d.ctl->done) return;
  const int i = blockIdx.x * MTHREADS + threadIdx.x;
  if (i >= d.TX) return;
  const int line = blockIdx.y;                       // k for the Y sweep, j for the Z sweep
  const int TL = DIR == 1 ? d.TY : d.TZ;
  const int c0 = blockIdx.z * CH, c1 = (c0 + CH < TL) ? c0 + CH : TL;   // cells this thread writes: [c0, c1)
  const long long str = DIR == 1 ? d.pitch : d.plane;
  const long long base = DIR == 1 ? d.id(i, 0, line) : d.id(i, line, 0);
  const T* __restrict__ vel = DIR == 1 ? A.st.vy : A.st.vz;
  const T dt = (T)d.ctl->dt;
  // per-line geometry factors (Tab. 5 products)
  const T gS = DIR == 1 ? d.syk[line] : d.szj[line];          // S = s^j s^k
  const T gV = DIR == 1 ? d.inv_syk[line] : d.invVj[line];    // 1/V = invVj / syk
  const T gL = DIR == 1 ? T(1) : d.Rzj[line];                 // LZ = dz R_z
  const T gD = DIR == 1 ? T(1) : d.invRzj[line];
  const T* __restrict__ tS = DIR == 1 ? d.syj : d.szk;
  const T* __restrict__ tV = DIR == 1 ? d.invVj : d.inv_syk;
  const T* __restrict__ tL = DIR == 1 ? d.LY : d.dz;
  const T* __restrict__ tD = DIR == 1 ? d.invDY : d.invdzc;

  // window: suffix 2 = cell r-2, 1 = cell r-1, 0 = cell r (just arrived), n = cell r+1 (in flight)
  T Q2[NQ + 1], Q1[NQ + 1], f2[NQ + 1], f1[NQ + 1], a2[NQ + 1], F2[NQ + 1];
#pragma unroll
  for (int q = 0; q <= NQ; ++q) { Q2[q] = Q1[q] = f2[q] = f1[q] = a2[q] = F2[q] = T(0); }
  T len2 = T(0), len1 = T(0), invd1 = T(0), w1 = T(0), S1 = T(0), dtiv2 = T(0), dtiv1 = T(0);

  T Qn[NQ + 1], wn = T(0);
  auto load_row = [&](const int r) {
    if (r >= 0 && r < TL) {
      const long long l = base + (long long)r * str;
      Qn[NQ] = A.srho[l];
#pragma unroll
      for (int q = 0; q < NQ; ++q) Qn[q] = A.sq[q][l];
      wn = vel[l];
    } else {
      Qn[NQ] = T(1);
#pragma unroll
      for (int q = 0; q < NQ; ++q) Qn[q] = T(0);
      wn = T(0);
    }
  };
  load_row(c0 - 2);
#pragma unroll 1
  for (int r = c0 - 2; r < c1 + 2; ++r) {
    // row r has arrived in Qn; start the loads of row r+1 at once
    T Q0[NQ + 1], f0[NQ + 1];
#pragma unroll
    for (int q = 0; q <= NQ; ++q) Q0[q] = Qn[q];
    const T w0 = wn;
    if (r + 1 < c1 + 2) load_row(r + 1);
    const int rc = r < 0 ? 0 : (r >= TL ? TL - 1 : r);
    const T len0 = DIR == 1 ? tL[rc] : tL[rc] * gL;
    const T invd0 = DIR == 1 ? tD[rc] : tD[rc] * gD;
    const T S0 = DIR == 1 ? tS[rc] * gS : gS * tS[rc];
    const T dtiv0 = dt * (DIR == 1 ? tV[rc] * gV : gV * tV[rc]);
    const T ir = T(1) / Q0[NQ];
#pragma unroll
    for (int q = 0; q < NQ; ++q) f0[q] = Q0[q] * ir;
    f0[NQ] = Q0[NQ];
    const int s = r - c0;   // stage of the pipeline (uniform over the block)
    T a1[NQ + 1], F1[NQ + 1];
#pragma unroll
    for (int q = 0; q <= NQ; ++q) { a1[q] = T(0); F1[q] = T(0); }
    if (s >= 0) {   // slopes of cell r-1
#pragma unroll
      for (int q = 0; q <= NQ; ++q) a1[q] = vl_slope(f2[q], f1[q], f0[q], invd1, invd0);
    }
    if (s >= 1) {   // fluxes through the lower face of cell r-1 (Eq. 48, Eqs. 45-47)
      const bool up = w1 >= T(0);
      const T wdt = w1 * dt;
      const T hup = (len2 - wdt) * T(0.5), hdn = (len1 + wdt) * T(0.5);
      const T rs = up ? f2[NQ] + a2[NQ] * hup : f1[NQ] - a1[NQ] * hdn;
      const T Fr = (w1 * rs) * S1;
      F1[NQ] = Fr;
#pragma unroll
      for (int q = 0; q < NQ; ++q) {
        const T fs = up ? f2[q] + a2[q] * hup : f1[q] - a1[q] * hdn;
        F1[q] = Fr * fs;
      }
    }
    if (s >= 2) {   // update (or pass through) cell r-2
      const int m = r - 2;
      const bool upd = m >= 2 && m < TL - 2;
      const long long l = base + (long long)m * str;
      A.drho[l] = upd ? Q2[NQ] - dtiv2 * (F1[NQ] - F2[NQ]) : Q2[NQ];
#pragma unroll
      for (int q = 0; q < NQ; ++q) A.dq[q][l] = upd ? Q2[q] - dtiv2 * (F1[q] - F2[q]) : Q2[q];
    }
#pragma unroll
    for (int q = 0; q <= NQ; ++q) { Q2[q] = Q1[q]; Q1[q] = Q0[q]; f2[q] = f1[q]; f1[q] = f0[q]; a2[q] = a1[q]; F2[q] = F1[q]; }
    len2 = len1; len1 = len0; invd1 = invd0; w1 = w0; S1 = S0; dtiv2 = dtiv1; dtiv1 = dtiv0;
  }
}

template <typename T, int NQ>
static int launch_sweep_nq(const Dev<T>& d, const SweepArgs<T>& a, int dir, cudaStream_t s) {
  if (dir == 0) {
    dim3 b(32, XW), g((d.TX + XIN - 1) / XIN, (d.TY + XW - 1) / XW, d.TZ);
    if (a.first) k_sweep_x<T, NQ, true><<<g, b, 0, s>>>(d, a);
    else k_sweep_x<T, NQ, false><<<g, b, 0, s>>>(d, a);
    return 1;
  }
  const int TL = dir == 1 ? d.TY : d.TZ, lines = dir == 1 ? d.TZ : d.TY;
  // chunk the sweep axis so that the grid fills the machine a few times over, but keep chunks long
  // (each one re-reads 4 rows of halo)
  const long long cols = (long long)((d.TX + MTHREADS - 1) / MTHREADS) * lines;
  int nch = (int)((148LL * 16 * 4 + cols - 1) / cols);
  if (nch < 1) nch = 1;
  int CH = (TL + nch - 1) / nch;
  if (CH < 32) CH = 32;
  if (CH > TL) CH = TL;
  nch = (TL + CH - 1) / CH;
  dim3 b(MTHREADS), g((d.TX + MTHREADS - 1) / MTHREADS, lines, nch);
  if (dir == 1) k_sweep_march<T, 1, NQ><<<g, b, 0, s>>>(d, a, CH);
  else k_sweep_march<T, 2, NQ><<<g, b, 0, s>>>(d, a, CH);
  return 1;
}

template <typename T>
int launch_sweep(const Dev<T>& d, const SweepArgs<T>& a, int dir, cudaStream_t s) {
  switch (a.nq) {
    case 2: return launch_sweep_nq<T, 2>(d, a, dir, s);
    case 3: return launch_sweep_nq<T, 3>(d, a, dir, s);
    case 4: return launch_sweep_nq<T, 4>(d, a, dir, s);
    case 5: return launch_sweep_nq<T, 5>(d, a, dir, s);
    case 6: return launch_sweep_nq<T, 6>(d, a, dir, s);
    case 7: return launch_sweep_nq<T, 7>(d, a, dir, s);
    default: return 0;
  }
}

template <typename T> void sweep_setup() {}
template void sweep_setup<double>();
template void sweep_setup<float>();

// ---- 12d: new velocities from the transported left/right momenta (Eq. 51), active cells ----------------
template <typename T>
__global__ void __launch_bounds__(128) k_newvel(const Dev<T> d, const T* __restrict__ rho, const QSet<T> S,
                                                const State<T> st) {
  if (d.ctl->done) return;
  const int ia = blockIdx.x * blockDim.x + threadIdx.x;
  if (ia >= d.nx) return;
  const int i = d.ngx + ia, j = d.ngy + blockIdx.y, k = d.ngz + blockIdx.z;
  const long long l = d.id(i, j, k);
  const T r0 = rho[l];
  if (d.hasx) {
    const T rx = d.Rx(j, k), rx2om = (rx * rx) * d.om_eff, irx = d.invRx(j, k);
    const long long lm = d.id(d.xw(i - 1), j, k);
    st.vx[l] = ((S.q[2][lm] + S.q[1][l]) / (rho[lm] + r0) - rx2om) * irx;
  }
  if (d.hasy) {
    const long long lm = l - d.pitch;
    st.vy[l] = (S.q[4][lm] + S.q[3][l]) / (rho[lm] + r0);
  }
  if (d.hasz) {
    const long long lm = l - d.plane;
    st.vz[l] = ((S.q[6][lm] + S.q[5][l]) / (rho[lm] + r0)) * d.invRzj[j];
  }
}

template <typename T>
int launch_newvel(const Dev<T>& d, const T* rho, const QSet<T>& set, const State<T>& st, cudaStream_t s) {
  dim3 b(128), g((d.nx + 127) / 128, d.ny, d.nz);
  k_newvel<T><<<g, b, 0, s>>>(d, rho, set, st);
  return 1;
}

#define INST(T)                                                                                    \
  template int launch_momenta<T>(const Dev<T>&, const State<T>&, const QSet<T>&, cudaStream_t);   \
  template int launch_sweep<T>(const Dev<T>&, const SweepArgs<T>&, int, cudaStream_t);             \
  template int launch_newvel<T>(const Dev<T>&, const T*, const QSet<T>&, const State<T>&, cudaStream_t);
INST(double)
INST(float)
#undef INST

}  // namespace fg
