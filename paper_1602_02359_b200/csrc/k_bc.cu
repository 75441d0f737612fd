// k_bc.cu -- ghost-zone boundary kernels (Fig. 2 cells 2 and 9).  Kinds: periodic
// (P:948), zero-gradient outflow, reflecting; formulas = DESIGN.md reading G22.
// Also the layout kernels (active cells <-> ghosted, padded arrays).
#include "kernels.h"

namespace fg {

// One thread per line (p,q) across the boundary direction; it walks the 3 ghost layers of every field
// in `mask` in the order stated in DESIGN.md (low/high side interleaved per layer), so that meshes
// thinner than the ghost depth behave as written there.
template <typename T, int DIR>
__global__ void k_bc(const Dev<T> d, const State<T> st, const int mask) {
  if (d.ctl->done) return;
  const int N = DIR == 0 ? d.nx : DIR == 1 ? d.ny : d.nz;
  const int ng = DIR == 0 ? d.ngx : DIR == 1 ? d.ngy : d.ngz;
  const int P = DIR == 0 ? d.TY : d.TX;
  const int Q = DIR == 2 ? d.TY : d.TZ;
  const int p = blockIdx.x * blockDim.x + threadIdx.x;
  const int q = blockIdx.y;
  if (p >= P || q >= Q) return;
  const long long base = DIR == 0 ? d.id(0, p, q) : DIR == 1 ? d.id(p, 0, q) : d.id(p, q, 0);
  const long long str = DIR == 0 ? 1 : DIR == 1 ? d.pitch : d.plane;
  const int m0 = ng, m1 = ng + N;
  const int lo = d.bc[DIR][0], hi = d.bc[DIR][1];
  T* const fields[5] = {st.rho, st.e, st.vx, st.vy, st.vz};
#pragma unroll
  for (int f = 0; f < 5; ++f) {
    if (!(mask & (1 << f))) continue;
    T* a = fields[f] + base;
    const bool normal = (f == 2 + DIR);
    for (int g = 0; g < ng; ++g) {
      if (lo == BC_PERIODIC) a[(m0 - 1 - g) * str] = a[(m1 - 1 - g) * str];
      else if (lo == BC_OUTFLOW) a[(m0 - 1 - g) * str] = a[m0 * str];
      else if (lo == BC_REFLECTING && !normal) a[(m0 - 1 - g) * str] = a[(m0 + g) * str];   // BC_EXTERNAL: left alone
      if (hi == BC_PERIODIC) a[(m1 + g) * str] = a[(m0 + g) * str];
      else if (hi == BC_OUTFLOW) a[(m1 + g) * str] = a[(m1 - 1) * str];
      else if (hi == BC_REFLECTING && !normal) a[(m1 + g) * str] = a[(m1 - 1 - g) * str];
    }
    if (normal && lo == BC_REFLECTING) {  // wall face at rest, velocity antisymmetric about it
      a[m0 * str] = T(0);
      for (int g = 1; g <= ng; ++g) a[(m0 - g) * str] = -a[(m0 + g) * str];
    }
    if (normal && hi == BC_REFLECTING) {
      a[m1 * str] = T(0);
      for (int g = 1; g <= ng - 1; ++g) a[(m1 + g) * str] = -a[(m1 - g) * str];
    }
  }
}

template <typename T>
int launch_bc(const Dev<T>& d, const State<T>& st, int mask, cudaStream_t s) {
  int n = 0;
  if (d.ngx > 0) {
    dim3 b(64), g((d.TY + 63) / 64, d.TZ);
    k_bc<T, 0><<<g, b, 0, s>>>(d, st, mask); ++n;
  }
  if (d.ngy > 0) {
    dim3 b(128), g((d.TX + 127) / 128, d.TZ);
    k_bc<T, 1><<<g, b, 0, s>>>(d, st, mask); ++n;
  }
  if (d.ngz > 0) {
    dim3 b(128), g((d.TX + 127) / 128, d.TY);
    k_bc<T, 2><<<g, b, 0, s>>>(d, st, mask); ++n;
  }
  return n;
}

// ---- layout kernels ---------------------------------------------------------------------------------
template <typename T>
__global__ void k_scatter(const Dev<T> d, const T* __restrict__ act, T* __restrict__ full) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y, k = blockIdx.z;
  if (i >= d.nx) return;
  full[d.id(i + d.ngx, j + d.ngy, k + d.ngz)] = act[(long long)i + (long long)d.nx * (j + (long long)d.ny * k)];
}
template <typename T>
__global__ void k_gather(const Dev<T> d, const T* __restrict__ full, T* __restrict__ act) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y, k = blockIdx.z;
  if (i >= d.nx) return;
  act[(long long)i + (long long)d.nx * (j + (long long)d.ny * k)] = full[d.id(i + d.ngx, j + d.ngy, k + d.ngz)];
}
template <typename T>
__global__ void k_unpad(const Dev<T> d, const T* __restrict__ full, T* __restrict__ out) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y, k = blockIdx.z;
  if (i >= d.TX) return;
  out[(long long)i + (long long)d.TX * (j + (long long)d.TY * k)] = full[d.id(i, j, k)];
}
template <typename T>
__global__ void k_copy(const Dev<T> d, const T* __restrict__ src, T* __restrict__ dst) {
  if (d.ctl->done) return;
  const long long n = d.narr;
  for (long long l = (long long)blockIdx.x * blockDim.x + threadIdx.x; l < n; l += (long long)gridDim.x * blockDim.x)
    dst[l] = src[l];
}

template <typename T>
int launch_scatter(const Dev<T>& d, const T* act, T* full, cudaStream_t s) {
  dim3 b(128), g((d.nx + 127) / 128, d.ny, d.nz);
  k_scatter<T><<<g, b, 0, s>>>(d, act, full);
  return 1;
}
template <typename T>
int launch_gather(const Dev<T>& d, const T* full, T* act, cudaStream_t s) {
  dim3 b(128), g((d.nx + 127) / 128, d.ny, d.nz);
  k_gather<T><<<g, b, 0, s>>>(d, full, act);
  return 1;
}
template <typename T>
int launch_unpad(const Dev<T>& d, const T* full, T* out, cudaStream_t s) {
  dim3 b(128), g((d.TX + 127) / 128, d.TY, d.TZ);
  k_unpad<T><<<g, b, 0, s>>>(d, full, out);
  return 1;
}
template <typename T>
int launch_copy(const Dev<T>& d, const T* src, T* dst, cudaStream_t s) {
  k_copy<T><<<148 * 8, 256, 0, s>>>(d, src, dst);
  return 1;
}

#define INST(T)                                                                          \
  template int launch_bc<T>(const Dev<T>&, const State<T>&, int, cudaStream_t);          \
  template int launch_scatter<T>(const Dev<T>&, const T*, T*, cudaStream_t);             \
  template int launch_gather<T>(const Dev<T>&, const T*, T*, cudaStream_t);              \
  template int launch_unpad<T>(const Dev<T>&, const T*, T*, cudaStream_t);               \
  template int launch_copy<T>(const Dev<T>&, const T*, T*, cudaStream_t);
INST(double)
INST(float)
#undef INST

}  // namespace fg
