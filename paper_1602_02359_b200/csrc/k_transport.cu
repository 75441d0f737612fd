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
  const T a = rdiv(T(2) * pr, den);
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
      const T rx = d.Rx(j, k), rx2om = d.xmom_off(j, rx), rz = d.Rzj[j];
      if (d.eos == EOS_ADI) mom[0] = A.st.e[l];
      mom[1] = r0 * rfma(rx, w, rx2om);
      mom[2] = r0 * rfma(rx, wp, rx2om);
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
  const T hup = rfma(-w, dt, len) * T(0.5), hdn = rfma(w, dt, len) * T(0.5);   // Eq. 48
  const T ir = rdiv(T(1), r0);

  // density: its mass flux F = w rho* S multiplies every other star value
  T Fr;
  {
    const T fm = shfl_up1(r0), fp = shfl_dn1(r0);
    const T a = vl_slope(fm, r0, fp, invd, invd);
    const T am = shfl_up1(a);
    const T rs = up ? rfma(am, hup, fm) : rfma(-a, hdn, r0);
    Fr = (w * rs) * Sm;
    const T Fp = shfl_dn1(Fr);
    if (inner) A.drho[l] = upd ? rfma(-dtiv, Fp - Fr, r0) : r0;
  }
#pragma unroll
  for (int q = 0; q < NQ; ++q) {
    const T f = Q[q] * ir;
    const T fm = shfl_up1(f), fp = shfl_dn1(f);
    const T a = vl_slope(fm, f, fp, invd, invd);
    const T am = shfl_up1(a);
    const T fs = up ? rfma(am, hup, fm) : rfma(-a, hdn, f);
    const T F = Fr * fs;
    const T Fp = shfl_dn1(F);
    if (inner) A.dq[q][l] = upd ? rfma(-dtiv, Fp - F, Q[q]) : Q[q];
  }
}

// ---- X sweep, two cells per lane ---------------------------------------------------------------------------
// A warp owns 64 consecutive cells of a row: lane L holds cells (t0 - 2 + 2L, +1) as one 16-byte vector
// per array.  Lanes 0 and 31 are the two-cell halo (recomputed, never stored), so a tile advances by 60
// cells.  Per quantity only four values cross lanes (f and the slope from the left, f and the flux from
// the right); everything else stays in registers.  The quantity list is fixed at compile time
// (e | pxm pxp | pym pyp | pzm pzp, Tab. 2) and the momenta are formed from the state on the fly (12a).
// Needs an even nx when X wraps (a pair never straddles the seam); odd rings take k_sweep_x.
template <typename T> struct Pair;
template <> struct Pair<double> { using type = double2; };
template <> struct Pair<float> { using type = float2; };

constexpr int X2W = 2;          // warps (rows) per block
constexpr int X2IN = 60;        // interior cells per warp

template <typename T>
__device__ __forceinline__ void ld_pair(const T* __restrict__ p, T& a, T& b) {
  const typename Pair<T>::type v = *reinterpret_cast<const typename Pair<T>::type*>(p);
  a = v.x; b = v.y;
}
template <typename T>
__device__ __forceinline__ void st_pair(T* __restrict__ p, const T a, const T b) {
  typename Pair<T>::type v; v.x = a; v.y = b;
  *reinterpret_cast<typename Pair<T>::type*>(p) = v;
}

template <typename T, bool ADI, bool HASY, bool HASZ, bool WRAP>
__global__ void __launch_bounds__(32 * X2W) k_sweep_x2(const Dev<T> d, const SweepArgs<T> A) {
  constexpr int NQ = (ADI ? 1 : 0) + 2 + (HASY ? 2 : 0) + (HASZ ? 2 : 0);
  if (d.ctl->done) return;
  const int lane = threadIdx.x;
  const int j = blockIdx.y * X2W + threadIdx.y, k = blockIdx.z;
  if (j >= d.TY) return;   // whole warps leave together
  const int iu = blockIdx.x * X2IN - 2 + 2 * lane;   // un-wrapped index of this lane's first cell
  int i = iu;
  bool have = true;
  if (WRAP) { i %= d.nx; if (i < 0) i += d.nx; }
  else have = iu >= 0 && iu < d.TX;   // the second cell of the pair may be row padding (never stored)
  const long long row = d.id(0, j, k);
  const long long l = row + (have ? i : 0);

  const T dt = (T)d.ctl->dt;
  const T len = d.LX(j, k), invd = d.invLX(j, k), Sm = d.Sx(j, k), dtiv = dt * d.invV(j, k);

  // ---- loads: everything this lane needs, issued up front ----
  T r[2] = {T(1), T(1)}, w[2] = {T(0), T(0)}, en[2] = {T(0), T(0)};
  T vy0[2] = {T(0), T(0)}, vy1[2] = {T(0), T(0)}, vz0[2] = {T(0), T(0)}, vz1[2] = {T(0), T(0)};
  if (have) {
    ld_pair(A.srho + l, r[0], r[1]);
    ld_pair(A.st.vx + l, w[0], w[1]);
    if (ADI) ld_pair(A.st.e + l, en[0], en[1]);
    if (HASY) {
      ld_pair(A.st.vy + l, vy0[0], vy0[1]);
      if (j + 1 < d.TY) ld_pair(A.st.vy + l + d.pitch, vy1[0], vy1[1]);
      else { vy1[0] = vy0[0]; vy1[1] = vy0[1]; }
    }
    if (HASZ) {
      ld_pair(A.st.vz + l, vz0[0], vz0[1]);
      if (k + 1 < d.TZ) ld_pair(A.st.vz + l + d.plane, vz1[0], vz1[1]);
      else { vz1[0] = vz0[0]; vz1[1] = vz0[1]; }
    }
  }
  // velocity on the upper face of the pair's second cell: the right neighbour's first, one extra load on lane 31
  T wn = shfl_dn1(w[0]);
  if (lane == 31 && have) {
    if (WRAP) { int ip = i + 2; if (ip >= d.nx) ip -= d.nx; wn = A.st.vx[row + ip]; }
    else if (i + 2 < d.TX) wn = A.st.vx[row + i + 2];
  }
  if (!WRAP) {   // the last cell of a ghosted row has no upper neighbour: its own face value stands in
    if (i + 2 >= d.TX) wn = w[1];
    if (i + 1 >= d.TX) w[1] = w[0];
  }

  // ---- 12a: the momenta of Tab. 2 ----
  T Q[NQ][2];
  {
    const T rx = d.Rx(j, k), rx2om = d.xmom_off(j, rx), rz = d.Rzj[j];
#pragma unroll
    for (int c = 0; c < 2; ++c) {
      const T wp = c == 0 ? w[1] : wn;
      int q = 0;
      if (ADI) Q[q++][c] = en[c];
      Q[q++][c] = r[c] * rfma(rx, w[c], rx2om);
      Q[q++][c] = r[c] * rfma(rx, wp, rx2om);
      if (HASY) { Q[q++][c] = r[c] * vy0[c]; Q[q++][c] = r[c] * vy1[c]; }
      if (HASZ) { Q[q++][c] = r[c] * (rz * vz0[c]); Q[q++][c] = r[c] * (rz * vz1[c]); }
    }
  }
  if (A.v0) { const T vm = A.v0[d.rid(j, k)]; w[0] = w[0] - vm; w[1] = w[1] - vm; }   // residual velocity
  bool up[2];
  T hup[2], hdn[2], ir[2];
#pragma unroll
  for (int c = 0; c < 2; ++c) {
    up[c] = w[c] >= T(0);                 // reading G3
    hup[c] = rfma(-w[c], dt, len) * T(0.5); hdn[c] = rfma(w[c], dt, len) * T(0.5);   // Eq. 48
    ir[c] = rdiv(T(1), r[c]);
  }
  const bool store = lane >= 1 && lane <= 30 && (WRAP ? iu < d.nx : have);

  // ---- density: its mass flux multiplies every other star value ----
  T Fr[2];
  {
    const T fl = shfl_up1(r[1]), fr = shfl_dn1(r[0]);
    const T a0 = vl_slope(fl, r[0], r[1], invd, invd);
    const T a1 = vl_slope(r[0], r[1], fr, invd, invd);
    const T al = shfl_up1(a1);
    const T s0 = up[0] ? rfma(al, hup[0], fl) : rfma(-a0, hdn[0], r[0]);
    const T s1 = up[1] ? rfma(a0, hup[1], r[0]) : rfma(-a1, hdn[1], r[1]);
    Fr[0] = (w[0] * s0) * Sm;
    Fr[1] = (w[1] * s1) * Sm;
    const T Fn = shfl_dn1(Fr[0]);
    {
      const T o0 = rfma(-dtiv, Fr[1] - Fr[0], r[0]), o1 = rfma(-dtiv, Fn - Fr[1], r[1]);
      if (WRAP) st2_if(A.drho + l, o0, o1, store);
      else {
        st_if(A.drho + l, (i >= 2 && i < d.TX - 2) ? o0 : r[0], store);
        st_if(A.drho + l + 1, (i + 1 >= 2 && i + 1 < d.TX - 2) ? o1 : r[1], store && i + 1 < d.TX);
      }
    }
  }
#pragma unroll
  for (int q = 0; q < NQ; ++q) {
    const T f0 = Q[q][0] * ir[0], f1 = Q[q][1] * ir[1];
    const T fl = shfl_up1(f1), fr = shfl_dn1(f0);
    const T a0 = vl_slope(fl, f0, f1, invd, invd);
    const T a1 = vl_slope(f0, f1, fr, invd, invd);
    const T al = shfl_up1(a1);
    const T s0 = up[0] ? rfma(al, hup[0], fl) : rfma(-a0, hdn[0], f0);
    const T s1 = up[1] ? rfma(a0, hup[1], f0) : rfma(-a1, hdn[1], f1);
    const T F0 = Fr[0] * s0, F1 = Fr[1] * s1;
    const T Fn = shfl_dn1(F0);
    {
      const T o0 = rfma(-dtiv, F1 - F0, Q[q][0]), o1 = rfma(-dtiv, Fn - F1, Q[q][1]);
      if (WRAP) st2_if(A.dq[q] + l, o0, o1, store);
      else {
        st_if(A.dq[q] + l, (i >= 2 && i < d.TX - 2) ? o0 : Q[q][0], store);
        st_if(A.dq[q] + l + 1, (i + 1 >= 2 && i + 1 < d.TX - 2) ? o1 : Q[q][1], store && i + 1 < d.TX);
      }
    }
  }
}

// ---- Y / Z sweep: marching with an asynchronous shared-memory ring -----------------------------------------
// One thread per (i, line) marches along the sweep axis; threads of a warp sit side by side along X, so
// every access is a coalesced row segment.  Rows are fetched RD rows ahead with cp.async into a ring of
// RS slots that is private to each thread (no barrier: a thread reads only what it copied itself), which
// keeps ~RD * (NQ+2) * 8 B per thread in flight without holding them in registers.  The ring also keeps
// rows r-1 and r-2, so the un-divided quantities of the cell being updated are re-read from shared
// memory instead of living in registers.  The row loop is unrolled by two so that the two-row window of
// q = Q / rho rotates by renaming.
#ifndef FG_MTHREADS
#define FG_MTHREADS 128
#define FG_MBLOCKS 3
#endif
constexpr int MTHREADS = FG_MTHREADS;
// Ring depth.  cp.async.ca passes through L1, and a line stays allocated there until its data has landed: the bytes a
// SM can keep in flight are bounded by the L1 that the shared-memory carve-out leaves.  With three blocks of 8 x 9 KB
// rings (221 KB) only 28 KB of L1 remain and the bare skeleton (no arithmetic) is capped at ~5.1 TB/s; with <= 196 KB of
// shared memory per SM (60 KB of L1) it moves 6.4 TB/s (profiles/r02a_marches.md).  So: as many slots as fit in
// 196 KB / blocks per SM, never more than 8; RS - 3 rows in flight (the ring also keeps rows r-1 and r-2).
__host__ __device__ constexpr int ring_slots(int na) {   // na: 8-byte words per cell and row; 8 KB per block go to the tables
  return (196 / FG_MBLOCKS - 8) / na < 8 ? (196 / FG_MBLOCKS - 8) / na : 8;
}

template <typename T> struct CpAsync;
template <> struct CpAsync<double> {
  static __device__ __forceinline__ void go(unsigned dst, const double* src) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dst), "l"(src) : "memory");
  }
};
template <> struct CpAsync<float> {
  static __device__ __forceinline__ void go(unsigned dst, const float* src) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(dst), "l"(src) : "memory");
  }
};
__device__ __forceinline__ void cp_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
// a load the compiler may not sink towards its use (volatile asm keeps its place among the cp.async statements)
__device__ __forceinline__ double ld_pinned(const double* p) {
  double v; asm volatile("ld.global.nc.f64 %0, [%1];" : "=d"(v) : "l"(p)); return v;
}
__device__ __forceinline__ float ld_pinned(const float* p) {
  float v; asm volatile("ld.global.nc.f32 %0, [%1];" : "=f"(v) : "l"(p)); return v;
}
template <int N> __device__ __forceinline__ void cp_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

template <typename T, int DIR, int NQ>
__global__ void __launch_bounds__(MTHREADS, FG_MBLOCKS) k_sweep_ring(const Dev<T> d, const SweepArgs<T> A, const int CH) {
  constexpr int NA = NQ + 2;   // rho, NQ quantities, the face velocity
  constexpr int RS = ring_slots(NA * (int)sizeof(T) / 8), RD = RS - 3;   // slots; rows in flight
  extern __shared__ __align__(16) unsigned char smem_raw[];
  T* const ring = reinterpret_cast<T*>(smem_raw) + threadIdx.x;   // element (slot, array) at (slot*NA + array)*MTHREADS
  if (d.ctl->done) return;
  int i = blockIdx.x * MTHREADS + threadIdx.x;
  const bool live = i < d.TX;
  if (!live) i = d.TX - 1;                            // idle lanes shadow the last column and store nothing
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

  const unsigned ring_s = (unsigned)__cvta_generic_to_shared(ring);
  const int nrow = (c1 - c0) + 4;                    // rows c0-2 .. c1+1, numbered n = 0 .. nrow-1
  // rows are taken in pairs without a test in between (a conditional second step costs ~60 register moves per pair where
  // the two paths merge): an odd chunk runs one row more, fetched like the others, which stores nothing
  const int nrow2 = (nrow + 1) & ~1;
  auto fetch = [&](const int n) {                    // row n -> slot n & (RS-1); rows off the array are clamped
    if (n < nrow2) {
      int r = c0 - 2 + n;
      r = r < 0 ? 0 : (r >= TL ? TL - 1 : r);
      const long long l = base + (long long)r * str;
      const unsigned dst = ring_s + (unsigned)(((n % RS) * NA) * MTHREADS * sizeof(T));
      CpAsync<T>::go(dst, A.srho + l);
#pragma unroll
      for (int q = 0; q < NQ; ++q) CpAsync<T>::go(dst + (unsigned)((1 + q) * MTHREADS * sizeof(T)), A.sq[q] + l);
      CpAsync<T>::go(dst + (unsigned)((NQ + 1) * MTHREADS * sizeof(T)), vel + l);
    }
    cp_commit();                                     // one group per row, empty past the end
  };
#pragma unroll
  for (int n = 0; n < RD; ++n) fetch(n);

  // window (index 0 = rho, 1..NQ = quantities): fA/fB hold q of rows r-2 / r-1 in turn, a2 the slope of
  // cell r-2, F2 the flux through the lower face of cell r-2
  T fA[NQ + 1], fB[NQ + 1], a2[NQ + 1], F2[NQ + 1];
#pragma unroll
  for (int q = 0; q <= NQ; ++q) { fA[q] = fB[q] = a2[q] = F2[q] = T(0); }
  T len2 = T(0), len1 = T(0), invd1 = T(0), w1 = T(0), S1 = T(0), dtiv2 = T(0), dtiv1 = T(0);

  // the geometry of the chunk's rows (Tab. 5 factors along the sweep axis), staged once in shared memory behind the ring:
  // a global load per row and table kept an LDG scoreboard busy in every row (ncu: a third of the long-scoreboard
  // stalls sat on the first FMA after it, profiles/r02b_final.md); a broadcast LDS has none of that
  T* const tab = reinterpret_cast<T*>(smem_raw) + (size_t)RS * NA * MTHREADS;   // [4][nrow2]
  for (int n = threadIdx.x; n < nrow2; n += MTHREADS) {
    const int r0 = c0 - 2 + n;
    const int rc = r0 < 0 ? 0 : (r0 >= TL ? TL - 1 : r0);
    tab[n] = tL[rc]; tab[nrow2 + n] = tD[rc]; tab[2 * nrow2 + n] = tS[rc]; tab[3 * nrow2 + n] = tV[rc];
  }
  __syncthreads();

  // one row: f2 (in: q of row r-2; out: q of row r), f1 (q of row r-1)
  auto row_step = [&](const int n, T (&f2)[NQ + 1], T (&f1)[NQ + 1]) {
    const int r = c0 - 2 + n;
    const T cL = tab[n], cD = tab[nrow2 + n], cS = tab[2 * nrow2 + n], cV = tab[3 * nrow2 + n];
    fetch(n + RD);
    cp_wait<RD>();                                   // row n has landed
    const T* cur = ring + ((n % RS) * NA) * MTHREADS;
    const T* old = ring + (((n + RS - 2) % RS) * NA) * MTHREADS;   // row r-2 (the cell being updated)
    const T len0 = DIR == 1 ? cL : cL * gL;
    const T invd0 = DIR == 1 ? cD : cD * gD;
    const T S0 = DIR == 1 ? cS * gS : gS * cS;
    const T dtiv0 = dt * (DIR == 1 ? cV * gV : gV * cV);
    const T w0 = cur[(NQ + 1) * MTHREADS];
    const T rho0 = cur[0];
    const T ir = rdiv(T(1), rho0);
    // face between cells r-2 and r-1 (Eq. 48, Eqs. 45-47)
    const bool up = w1 >= T(0);
    const T hup = rfma(-w1, dt, len2) * T(0.5), hdn = rfma(w1, dt, len1) * T(0.5);
    const int m = r - 2;
    const bool wr = n >= 4 && n < nrow && live;
    const bool upd = m >= 2 && m < TL - 2;
    const long long lo = base + (long long)m * str;
    T Fr;
    {
      const T f0 = rho0;
      const T a1 = vl_slope(f2[0], f1[0], f0, invd1, invd0);
      const T rs = up ? rfma(a2[0], hup, f2[0]) : rfma(-a1, hdn, f1[0]);
      Fr = (w1 * rs) * S1;
      { const T Qo = old[0]; st_if(A.drho + lo, upd ? rfma(-dtiv2, Fr - F2[0], Qo) : Qo, wr); }
      f2[0] = f0; a2[0] = a1; F2[0] = Fr;
    }
#pragma unroll
    for (int q = 1; q <= NQ; ++q) {
      const T f0 = cur[q * MTHREADS] * ir;
      const T a1 = vl_slope(f2[q], f1[q], f0, invd1, invd0);
      const T fs = up ? rfma(a2[q], hup, f2[q]) : rfma(-a1, hdn, f1[q]);
      const T F1 = Fr * fs;
      { const T Qo = old[q * MTHREADS]; st_if(A.dq[q - 1] + lo, upd ? rfma(-dtiv2, F1 - F2[q], Qo) : Qo, wr); }
      f2[q] = f0; a2[q] = a1; F2[q] = F1;
    }
    len2 = len1; len1 = len0; invd1 = invd0; w1 = w0; S1 = S0; dtiv2 = dtiv1; dtiv1 = dtiv0;
  };
#pragma unroll 1
  for (int n = 0; n < nrow2; n += 2) {
    row_step(n, fA, fB);
    row_step(n + 1, fB, fA);
  }
  cp_wait<0>();
}

template <typename T, bool ADI, bool HASY, bool HASZ>
static int launch_x2(const Dev<T>& d, const SweepArgs<T>& a, cudaStream_t s) {
  const int span = d.xwrap ? d.nx : d.TX;
  dim3 b(32, X2W), g((span + X2IN - 1) / X2IN, (d.TY + X2W - 1) / X2W, d.TZ);
  if (d.xwrap) k_sweep_x2<T, ADI, HASY, HASZ, true><<<g, b, 0, s>>>(d, a);
  else k_sweep_x2<T, ADI, HASY, HASZ, false><<<g, b, 0, s>>>(d, a);
  return 1;
}

template <typename T, int NQ>
static int launch_sweep_nq(const Dev<T>& d, const SweepArgs<T>& a, int dir, cudaStream_t s) {
  if (dir == 0) {   // the X sweep is always the first pass: 12a is fused into it
    if (!d.xwrap || d.nx % 2 == 0) {
      const int key = (d.eos == EOS_ADI ? 4 : 0) | (d.hasy ? 2 : 0) | (d.hasz ? 1 : 0);
      switch (key) {
        case 0: return launch_x2<T, false, false, false>(d, a, s);
        case 1: return launch_x2<T, false, false, true>(d, a, s);
        case 2: return launch_x2<T, false, true, false>(d, a, s);
        case 3: return launch_x2<T, false, true, true>(d, a, s);
        case 4: return launch_x2<T, true, false, false>(d, a, s);
        case 5: return launch_x2<T, true, false, true>(d, a, s);
        case 6: return launch_x2<T, true, true, false>(d, a, s);
        default: return launch_x2<T, true, true, true>(d, a, s);
      }
    }
    dim3 b(32, XW), g((d.TX + XIN - 1) / XIN, (d.TY + XW - 1) / XW, d.TZ);
    k_sweep_x<T, NQ, true><<<g, b, 0, s>>>(d, a);
    return 1;
  }
  const int TL = dir == 1 ? d.TY : d.TZ, lines = dir == 1 ? d.TZ : d.TY;
  // chunk the sweep axis: equal blocks run in rounds of the resident slots; each chunk re-reads 4 rows of halo
  const long long cols = (long long)((d.TX + MTHREADS - 1) / MTHREADS) * lines;
  const size_t ring = (size_t)ring_slots((NQ + 2) * (int)sizeof(T) / 8) * (NQ + 2) * MTHREADS * sizeof(T);
  static int slots = 0;   // per instantiation (T, NQ): the two directions have the same resources
  if (!slots) slots = resident_slots(k_sweep_ring<T, 1, NQ>, MTHREADS, ring + 4096);
  int CH = pick_chunk_len(cols, TL, 4, slots, 16);
  if (CH > 216) CH = 216;                                   // the chunk's geometry tables sit behind the ring: 4 x (CH + 5) reals, <= 7 KB
  const int nch = (TL + CH - 1) / CH;
  const size_t sm = ring + (size_t)4 * (CH + 5) * sizeof(T);
  dim3 b(MTHREADS), g((d.TX + MTHREADS - 1) / MTHREADS, lines, nch);
  if (dir == 1) k_sweep_ring<T, 1, NQ><<<g, b, sm, s>>>(d, a, CH);
  else k_sweep_ring<T, 2, NQ><<<g, b, sm, s>>>(d, a, CH);
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

template <typename T, int NQ> static void ring_attr() {
  const int sm = ring_slots((NQ + 2) * (int)sizeof(T) / 8) * (NQ + 2) * MTHREADS * (int)sizeof(T) + 4 * 221 * (int)sizeof(T);
  cudaFuncSetAttribute(k_sweep_ring<T, 1, NQ>, cudaFuncAttributeMaxDynamicSharedMemorySize, sm);
  cudaFuncSetAttribute(k_sweep_ring<T, 2, NQ>, cudaFuncAttributeMaxDynamicSharedMemorySize, sm);
  // no carve-out request: the driver then picks the smallest shared-memory configuration that holds the resident blocks
  // (196 KB here) and L1 keeps the rest; asking for 86 % or 100 % was measured to select the 228 KB one (see ring_slots)
}
template <typename T> void sweep_setup() {
  ring_attr<T, 2>(); ring_attr<T, 3>(); ring_attr<T, 4>(); ring_attr<T, 5>(); ring_attr<T, 6>(); ring_attr<T, 7>();
}

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
    const T rx = d.Rx(j, k), rx2om = d.xmom_off(j, rx), irx = d.invRx(j, k);
    const long long lm = d.id(d.xw(i - 1), j, k);
    st.vx[l] = (rdiv(S.q[2][lm] + S.q[1][l], rho[lm] + r0) - rx2om) * irx;
  }
  if (d.hasy) {
    const long long lm = l - d.pitch;
    st.vy[l] = rdiv(S.q[4][lm] + S.q[3][l], rho[lm] + r0);
  }
  if (d.hasz) {
    const long long lm = l - d.plane;
    st.vz[l] = rdiv(S.q[6][lm] + S.q[5][l], rho[lm] + r0) * d.invRzj[j];
  }
}

template <typename T>
int launch_newvel(const Dev<T>& d, const T* rho, const QSet<T>& set, const State<T>& st, cudaStream_t s) {
  dim3 b(128), g((d.nx + 127) / 128, d.ny, d.nz);
  k_newvel<T><<<g, b, 0, s>>>(d, rho, set, st);
  return 1;
}

// ---- 12d + cell 6 of the NEXT update: Eq. 51, then the CFL rate of the new state -------------------------------
// Meshes without orbital advection, X wrapped, Y and Z periodic.  The cell's new velocities are stored as k_newvel
// stores them; the velocities on its three upper faces are re-formed from the neighbours' momenta (one division
// each), with the index the periodic ghost fill of the next update would copy from, and the per-cell rate of
// Eq. 59 (same expressions as k_dt_cells) goes into the running max that k_dt_finish of the next update turns into
// dt.  The dt pass (40 B per cell) disappears; newvel reads e in addition (88 B per cell instead of 80 + 40).
template <typename T, bool ADI>
__global__ void __launch_bounds__(128) k_newvel_dt(const Dev<T> d, const T* __restrict__ rho, const T* __restrict__ en,
                                                   const QSet<T> S, const State<T> st) {
  if (d.ctl->done) return;
  const int ia = blockIdx.x * blockDim.x + threadIdx.x;
  const bool live = ia < d.nx;
  const int i = live ? ia : 0, j = d.ngy + blockIdx.y, k = d.ngz + blockIdx.z;
  const long long row = d.id(0, j, k), l = row + i;
  const long long lxm = row + (i == 0 ? d.nx - 1 : i - 1), lxp = row + (i + 1 == d.nx ? 0 : i + 1);
  // upper neighbours in Y and Z: where the periodic ghost fill takes the face value from
  const int jp = j + 1 == d.ngy + d.ny ? d.ngy : j + 1, kp = k + 1 == d.ngz + d.nz ? d.ngz : k + 1;
  const long long lyp = d.id(i, jp, k), lzp = d.id(i, j, kp);
  const T r0 = rho[l];
  const T rx = d.Rx(j, k), rx2om = d.xmom_off(j, rx), irx = d.invRx(j, k), irz = d.invRzj[j];
  // Eq. 51 on the three lower faces (stored) ...
  const T ax = (rdiv(S.q[2][lxm] + S.q[1][l], rho[lxm] + r0) - rx2om) * irx;
  const T ay = rdiv(S.q[4][l - d.pitch] + S.q[3][l], rho[l - d.pitch] + r0);
  const T az = rdiv(S.q[6][l - d.plane] + S.q[5][l], rho[l - d.plane] + r0) * irz;
  // ... and on the three upper faces: the neighbours' own values.  X: the next lane's (re-formed at the end of the
  // warp and of the ring); Y, Z: re-formed from this cell's and the upper neighbour's momenta, or, on the last active
  // row / plane, at the index the periodic ghost fill copies from
  T bx = __shfl_down_sync(0xffffffffu, ax, 1);
  if ((threadIdx.x & 31) == 31 || i + 1 >= d.nx) bx = (rdiv(S.q[2][l] + S.q[1][lxp], r0 + rho[lxp]) - rx2om) * irx;
  const bool wy = jp != j + 1, wz = kp != k + 1;   // uniform over the block
  const T by = rdiv((wy ? S.q[4][lyp - d.pitch] : S.q[4][l]) + S.q[3][lyp], (wy ? rho[lyp - d.pitch] : r0) + rho[lyp]);
  const T bz = rdiv((wz ? S.q[6][lzp - d.plane] : S.q[6][l]) + S.q[5][lzp], (wz ? rho[lzp - d.plane] : r0) + rho[lzp]) * irz;
  if (live) { st.vx[l] = ax; st.vy[l] = ay; st.vz[l] = az; }
  // Eq. 59 for the new state
  const T ilx = d.invLX(j, k), ily = d.invLY[j], ilz = d.invLZ(j, k);
  const T ilmax = rmax(rmax(rmax(T(0), ilx), ily), ilz);
  const T il2 = ilmax * ilmax;
  const T I4 = d.c4 * il2;
  const T e0 = en[l];
  const T cs2 = ADI ? rdiv(d.gg1 * e0, r0) : e0 * e0;
  const T I1sq = cs2 * il2;
  T I2 = T(0), I3 = T(0);
  I2 = rmax(I2, rabs(T(0.5) * (ax + bx)) * ilx);
  I3 = rmax(I3, rabs(bx - ax) * ilx);
  I2 = rmax(I2, rabs(T(0.5) * (ay + by)) * ily);
  I3 = rmax(I3, rabs(by - ay) * ily);
  I2 = rmax(I2, rabs(T(0.5) * (az + bz)) * ilz);
  I3 = rmax(I3, rabs(bz - az) * ilz);
  I3 = d.c3 * I3;
  T m2 = live ? rfma(I4, I4, rfma(I3, I3, rfma(I2, I2, I1sq))) : T(0);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) m2 = rmax(m2, __shfl_xor_sync(0xffffffffu, m2, o));
  __shared__ T sm[4];
  if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = m2;
  __syncthreads();
  if (threadIdx.x == 0) {
    m2 = rmax(rmax(sm[0], sm[1]), rmax(sm[2], sm[3]));
    // a million blocks, one address: only a block that raises the running max pays for the atomic
    const unsigned long long b = to_bits(m2);
    if (b > *(volatile unsigned long long*)&d.ctl->m2bits) atomicMax(&d.ctl->m2bits, b);
  }
}

// The same with TWO cells per lane (even nx): 16-byte accesses, the X neighbours by shuffle (lanes 0 and 31 of a warp
// load their outer neighbour), half the address arithmetic and twice the loads in flight per thread.  Every expression
// is the one k_newvel_dt evaluates for the same face, so the results are bit-identical.
// Blocks of 64 threads (128 cells) and no register cap: at 512^3 that is 2.30 ms against 2.61 with 128 threads (66
// registers), 2.62 with 96, and 3.1-3.4 ms for every variant whose registers were capped by a minimum block count
// (ptxas then sinks half of the loads behind the arithmetic); tiles of 2-8 rows x 64 cells cost 2.9-3.4 ms
// (profiles/r02b_final.md).
constexpr int NVT = 64;
template <typename T, bool ADI>
__global__ void __launch_bounds__(NVT) k_newvel_dt2(const Dev<T> d, const T* __restrict__ rho, const T* __restrict__ en,
                                                    const QSet<T> S, const State<T> st) {
  if (d.ctl->done) return;
  const int ia = 2 * (blockIdx.x * blockDim.x + threadIdx.x);
  const bool live = ia < d.nx;
  const int i = live ? ia : 0, j = d.ngy + blockIdx.y, k = d.ngz + blockIdx.z;
  const int lane = threadIdx.x & 31;
  const long long row = d.id(0, j, k), l = row + i;
  const int jp = j + 1 == d.ngy + d.ny ? d.ngy : j + 1, kp = k + 1 == d.ngz + d.nz ? d.ngz : k + 1;
  const long long lyp = d.id(i, jp, k), lzp = d.id(i, j, kp);
  const bool wy = jp != j + 1, wz = kp != k + 1;   // uniform over the block
  const T rx = d.Rx(j, k), rx2om = d.xmom_off(j, rx), irx = d.invRx(j, k), irz = d.invRzj[j];
  T r0[2], xm[2], xp[2], ym[2], zm[2], e0[2];
  ld_pair(rho + l, r0[0], r0[1]);
  ld_pair(S.q[1] + l, xm[0], xm[1]);
  ld_pair(S.q[2] + l, xp[0], xp[1]);
  ld_pair(S.q[3] + l, ym[0], ym[1]);
  ld_pair(S.q[5] + l, zm[0], zm[1]);
  ld_pair(en + l, e0[0], e0[1]);
  T ryl[2], ypl[2], rzl[2], zpl[2];              // lower neighbours in Y and Z
  ld_pair(rho + l - d.pitch, ryl[0], ryl[1]);
  ld_pair(S.q[4] + l - d.pitch, ypl[0], ypl[1]);
  ld_pair(rho + l - d.plane, rzl[0], rzl[1]);
  ld_pair(S.q[6] + l - d.plane, zpl[0], zpl[1]);
  T ryu[2], ymu[2], ypc[2], ryc[2], rzu[2], zmu[2], zpc[2], rzc[2];   // upper faces: neighbour's own operands
  ld_pair(rho + lyp, ryu[0], ryu[1]);
  ld_pair(S.q[3] + lyp, ymu[0], ymu[1]);
  ld_pair(rho + lzp, rzu[0], rzu[1]);
  ld_pair(S.q[5] + lzp, zmu[0], zmu[1]);
  if (wy) { ld_pair(S.q[4] + lyp - d.pitch, ypc[0], ypc[1]); ld_pair(rho + lyp - d.pitch, ryc[0], ryc[1]); }
  else { ld_pair(S.q[4] + l, ypc[0], ypc[1]); ryc[0] = r0[0]; ryc[1] = r0[1]; }
  if (wz) { ld_pair(S.q[6] + lzp - d.plane, zpc[0], zpc[1]); ld_pair(rho + lzp - d.plane, rzc[0], rzc[1]); }
  else { ld_pair(S.q[6] + l, zpc[0], zpc[1]); rzc[0] = r0[0]; rzc[1] = r0[1]; }
  // X neighbours: the pair to the left gives (rho, pxp) of cell i-1, the pair to the right (rho, pxm) of cell i+2
  T rl = shfl_up1(r0[1]), pl = shfl_up1(xp[1]), rr = shfl_dn1(r0[0]), pr = shfl_dn1(xm[0]);
  if (lane == 0 || i == 0) { const long long lm = row + (i == 0 ? d.nx - 1 : i - 1); rl = rho[lm]; pl = S.q[2][lm]; }
  if (lane == 31 || i + 2 >= d.nx) { const long long lq = row + (i + 2 >= d.nx ? 0 : i + 2); rr = rho[lq]; pr = S.q[1][lq]; }
  // Eq. 51 on the lower faces of both cells and on the upper X face of the second
  const T ax0 = (rdiv(pl + xm[0], rl + r0[0]) - rx2om) * irx;
  const T ax1 = (rdiv(xp[0] + xm[1], r0[0] + r0[1]) - rx2om) * irx;
  const T ax2 = (rdiv(xp[1] + pr, r0[1] + rr) - rx2om) * irx;
  T ay[2], az[2], by[2], bz[2];
#pragma unroll
  for (int c = 0; c < 2; ++c) {
    ay[c] = rdiv(ypl[c] + ym[c], ryl[c] + r0[c]);
    az[c] = rdiv(zpl[c] + zm[c], rzl[c] + r0[c]) * irz;
    by[c] = rdiv(ypc[c] + ymu[c], ryc[c] + ryu[c]);
    bz[c] = rdiv(zpc[c] + zmu[c], rzc[c] + rzu[c]) * irz;
  }
  if (live) { st_pair(st.vx + l, ax0, ax1); st_pair(st.vy + l, ay[0], ay[1]); st_pair(st.vz + l, az[0], az[1]); }
  // Eq. 59 for the new state
  const T ilx = d.invLX(j, k), ily = d.invLY[j], ilz = d.invLZ(j, k);
  const T ilmax = rmax(rmax(rmax(T(0), ilx), ily), ilz);
  const T il2 = ilmax * ilmax;
  const T I4 = d.c4 * il2;
  T m2 = T(0);
#pragma unroll
  for (int c = 0; c < 2; ++c) {
    const T cs2 = ADI ? rdiv(d.gg1 * e0[c], r0[c]) : e0[c] * e0[c];
    const T I1sq = cs2 * il2;
    const T ax = c ? ax1 : ax0, bx = c ? ax2 : ax1;
    T I2 = T(0), I3 = T(0);
    I2 = rmax(I2, rabs(T(0.5) * (ax + bx)) * ilx);
    I3 = rmax(I3, rabs(bx - ax) * ilx);
    I2 = rmax(I2, rabs(T(0.5) * (ay[c] + by[c])) * ily);
    I3 = rmax(I3, rabs(by[c] - ay[c]) * ily);
    I2 = rmax(I2, rabs(T(0.5) * (az[c] + bz[c])) * ilz);
    I3 = rmax(I3, rabs(bz[c] - az[c]) * ilz);
    I3 = d.c3 * I3;
    if (live) m2 = rmax(m2, rfma(I4, I4, rfma(I3, I3, rfma(I2, I2, I1sq))));
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) m2 = rmax(m2, __shfl_xor_sync(0xffffffffu, m2, o));
  __shared__ T sm[NVT / 32];
  if (lane == 0) sm[threadIdx.x >> 5] = m2;
  __syncthreads();
  if (threadIdx.x == 0) {
#pragma unroll
    for (int n = 1; n < NVT / 32; ++n) m2 = rmax(m2, sm[n]);
    const unsigned long long b = to_bits(m2);
    if (b > *(volatile unsigned long long*)&d.ctl->m2bits) atomicMax(&d.ctl->m2bits, b);
  }
}

template <typename T>
bool newvel_dt_ok(const Dev<T>& d) {
  return d.hasx && d.hasy && d.hasz && d.xwrap && !d.fargo && d.bc[1][0] == BC_PERIODIC && d.bc[1][1] == BC_PERIODIC &&
         d.bc[2][0] == BC_PERIODIC && d.bc[2][1] == BC_PERIODIC;
}

template <typename T>
int launch_newvel_dt(const Dev<T>& d, const T* rho, const T* en, const QSet<T>& set, const State<T>& st, cudaStream_t s) {
  if (d.nx % 2 == 0) {
    dim3 b(NVT), g((d.nx / 2 + NVT - 1) / NVT, d.ny, d.nz);
    if (d.eos == EOS_ADI) k_newvel_dt2<T, true><<<g, b, 0, s>>>(d, rho, en, set, st);
    else k_newvel_dt2<T, false><<<g, b, 0, s>>>(d, rho, en, set, st);
    return 1;
  }
  dim3 b(128), g((d.nx + 127) / 128, d.ny, d.nz);
  if (d.eos == EOS_ADI) k_newvel_dt<T, true><<<g, b, 0, s>>>(d, rho, en, set, st);
  else k_newvel_dt<T, false><<<g, b, 0, s>>>(d, rho, en, set, st);
  return 1;
}

#define INST(T)                                                                                    \
  template int launch_momenta<T>(const Dev<T>&, const State<T>&, const QSet<T>&, cudaStream_t);   \
  template int launch_sweep<T>(const Dev<T>&, const SweepArgs<T>&, int, cudaStream_t);             \
  template int launch_newvel<T>(const Dev<T>&, const T*, const QSet<T>&, const State<T>&, cudaStream_t);       \
  template bool newvel_dt_ok<T>(const Dev<T>&);                                                              \
  template int launch_newvel_dt<T>(const Dev<T>&, const T*, const T*, const QSet<T>&, const State<T>&, cudaStream_t);
INST(double)
INST(float)
#undef INST

}  // namespace fg
