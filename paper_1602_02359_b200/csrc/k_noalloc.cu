// fargo_diagnostics_noalloc (include/fargo.h): the sum reductions of P:787 ("the mass or angular momentum") for callers
// that cannot allocate -- code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.
//
// The existing path (fargo_diagnostics) writes one partial sum per block into a region of the caller's workspace, copies
// the partials to a host vector and adds them there.  This variant keeps the partials in a file-scope device array of
// fixed size, adds them ON THE DEVICE in the same (block) order, and writes the five sums to a DEVICE address the caller
// owns.  It calls no cudaMalloc / cudaFree / cudaMallocHost, builds no host container and does not synchronise.
//
//   * g_na_part holds NA_MAX_BLOCKS x 5 doubles = 2.5 MiB on every device that loads the library, until exit.
//   * One block reduces 8 rings (rows along X), so a mesh fits when ceil(ny * nz / 8) <= NA_MAX_BLOCKS, i.e.
//     ny * nz <= 524288 (512 x 512 and 724 x 724 fit); larger meshes are rejected with an error, never truncated.
//   * Every call on a device shares the one array.  Nothing in it has to start at zero: each block of a call overwrites
//     its own five partials before the finishing kernel reads exactly the blocks of that call, so the contents left by
//     the previous call (of this or another context) are never read.  Two calls that OVERLAP on the GPU (different
//     streams, no dependency) race on the array: order them.
//   * In host code `g_na_part` is the host-side stand-in of the symbol, not a device address.  The address handed to the
//     kernels comes from cudaGetSymbolAddress, looked up once per device with that device current (na_scratch below);
//     the first call on a device therefore loads the module if the driver had not yet done so -- make it once before a
//     graph capture.
#include <mutex>
#include <string>

#include "common.cuh"
#include "kernels.h"

namespace fg {

constexpr int NA_MAX_BLOCKS = 65536;      // blocks of k_diagnostics whose partials fit (8 rings each)
constexpr int NA_MAX_DEVICES = 64;
static __device__ __align__(256) double g_na_part[(size_t)NA_MAX_BLOCKS * 5];

// rings (rows along X) that one block of k_diagnostics reduces: read off planets_blocks(), which owns that number
static int na_rings_per_block() {
  int per = 1;
  while (planets_blocks(per + 1, 1) == 1) ++per;
  return per;
}
long long diagnostics_noalloc_max_rings() { return (long long)NA_MAX_BLOCKS * na_rings_per_block(); }

// out[c] = part[0][c] + part[1][c] + ... in block order: the order in which fargo_diagnostics adds them on the host, so
// both paths round alike.  Five threads, one chain of additions each; the loads of a batch are independent and overlap.
__global__ void __launch_bounds__(32) k_diag_finish(const double* __restrict__ part, const int nblk, double* __restrict__ out) {
  const int c = threadIdx.x;
  if (c >= 5) return;
  double s = 0.0;
  int b = 0;
  for (; b + 8 <= nblk; b += 8) {
    double v[8];
#pragma unroll
    for (int u = 0; u < 8; ++u) v[u] = part[(size_t)(b + u) * 5 + c];
#pragma unroll
    for (int u = 0; u < 8; ++u) s = s + v[u];
  }
  for (; b < nblk; ++b) s = s + part[(size_t)b * 5 + c];
  out[c] = s;
}

// device address of g_na_part on the CURRENT device (looked up once per device); nullptr + message on failure
static double* na_scratch(std::string& err) {
  static std::mutex mu;
  static double* ptr[NA_MAX_DEVICES] = {};
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) { err = std::string("cudaGetDevice: ") + cudaGetErrorString(e); return nullptr; }
  if (dev < 0 || dev >= NA_MAX_DEVICES) { err = "device ordinal beyond the table of fargo_diagnostics_noalloc"; return nullptr; }
  std::lock_guard<std::mutex> lock(mu);
  if (!ptr[dev]) {
    double* p = nullptr;
    e = cudaGetSymbolAddress((void**)&p, g_na_part);
    if (e != cudaSuccess || !p) {
      err = std::string("cudaGetSymbolAddress(g_na_part): ") + cudaGetErrorString(e);
      return nullptr;
    }
    ptr[dev] = p;
  }
  return ptr[dev];
}

// Launches on `s`: k_diagnostics (the kernel of fargo_diagnostics, its partials in g_na_part) and k_diag_finish.
// Returns the number of launches, or -1 (size beyond the maximum) / -2 (CUDA error) with `err` set.
template <typename T>
int launch_diagnostics_noalloc(const Dev<T>& d, const State<T>& st, double* out_device, cudaStream_t s, std::string& err) {
  const long long rings = (long long)d.ny * d.nz;
  const long long nblk = planets_blocks(d.ny, d.nz);
  if (nblk > NA_MAX_BLOCKS) {
    err = "fargo_diagnostics_noalloc: ny * nz = " + std::to_string(rings) + " rings need " + std::to_string(nblk) +
          " partial-sum blocks, the static scratch holds " + std::to_string(NA_MAX_BLOCKS) + " (ny * nz <= " +
          std::to_string(diagnostics_noalloc_max_rings()) + "); use fargo_diagnostics";
    return -1;
  }
  double* part = na_scratch(err);
  if (!part) return -2;
  int n = launch_diagnostics<T>(d, st, part, s);
  k_diag_finish<<<1, 32, 0, s>>>(part, (int)nblk, out_device);
  return n + 1;
}

template int launch_diagnostics_noalloc<double>(const Dev<double>&, const State<double>&, double*, cudaStream_t, std::string&);
template int launch_diagnostics_noalloc<float>(const Dev<float>&, const State<float>&, double*, cudaStream_t, std::string&);

}  // namespace fg
