// gk_noalloc.cu -- gk_spectra_static (include/gk.h): the spectra of |phi|^2 for callers that cannot allocate.
//
// Who this is for.  gk_spectra needs a gk_ctx, and gk_create fills that context with cudaMalloc'ed tables and a
// staging block.  Some hosts of this library cannot do that: a diagnostics hook inside an application whose own pool
// allocator (a framework's caching allocator, RMM, a preallocating runtime) has already taken the whole device, so
// that any further cudaMalloc fails; a process pinned under an MPS / MIG memory cap; a latency-critical loop in which
// cudaMalloc's implicit device-wide synchronisation is not acceptable.  Such a caller already holds phi on the device
// (from its own solver, or from gk_field_solve of a context somebody else created) and only wants the two spectra.
//
// What it does differently.  The kernel is gk_spectra_kernel's summation (gk_kernels.cuh: one block per output, one
// deterministic tree, double accumulation -- same order, so the same bits) with the grid sizes as plain integers and
// the device-side staging of the nkx + nky results in a fixed array that lives in the library image instead of in a
// context.  Nothing here calls cudaMalloc, cudaFree, or a library routine that allocates; the host side keeps its
// error text in a fixed thread-local buffer.
//
// What that costs.  Every GPU that loads libgk.so holds GK_SPECTRA_STATIC_MAX doubles (32 KiB) until the process
// exits, and ALL calls on a device share that one array: two calls that overlap on the GPU (different streams, or
// different host threads) race on it.  The array keeps the previous call's numbers; every call overwrites the
// nkx + nky entries it reads back and reads no other, so nothing has to be cleared first.
#include <cstdarg>
#include <cstdio>
#include <mutex>

#include <cuda_runtime.h>

#include "../../include/gk.h"

namespace {

constexpr int kMaxOut = GK_SPECTRA_STATIC_MAX;   // most outputs (nkx + nky) one call may ask for
constexpr int kMaxDev = 64;                      // devices a process can address through this entry point

// The scratch.  In host code this NAME is only a host-side shadow of the symbol, not a device address: it must
// never be handed to a kernel or to cudaMemcpy as a pointer.  Host code gets the real per-device address from
// cudaGetSymbolAddress (scratch_for_current_device below); device code could name it directly.
static __device__ __align__(256) double g_spec_scratch[kMaxOut];

std::mutex g_mu;
double *g_scratch_addr[kMaxDev];   // device address of g_spec_scratch on device d, resolved on first use there

thread_local char t_err[256] = "";

int reject(int code, const char *fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(t_err, sizeof(t_err), fmt, ap);
  va_end(ap);
  return code;
}

// Set-up, once per device, with that device current: resolves the address of this device's copy of the array.
int scratch_for_current_device(double **out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return reject(GK_ECUDA, "gk_spectra_static: cudaGetDevice: %s", cudaGetErrorString(e));
  if (dev < 0 || dev >= kMaxDev) return reject(GK_EUNSUPPORTED, "gk_spectra_static: device ordinal %d beyond %d", dev, kMaxDev - 1);
  std::lock_guard<std::mutex> lock(g_mu);
  if (!g_scratch_addr[dev]) {
    void *p = nullptr;
    e = cudaGetSymbolAddress(&p, g_spec_scratch);
    if (e != cudaSuccess || !p)
      return reject(GK_ECUDA, "gk_spectra_static: cudaGetSymbolAddress on device %d: %s", dev, cudaGetErrorString(e));
    g_scratch_addr[dev] = (double *)p;
  }
  *out = g_scratch_addr[dev];
  return GK_OK;
}

// PAPER.md:113, 390 (reading R20), as gk::gk_spectra_kernel: block b < nkx sums row p = b over (s, ky) with the
// Parseval factor (1 at ky = 0, 2 otherwise); block nkx + m sums column m over (s, kx); weight 1/ns.
__global__ void __launch_bounds__(256) gk_spectra_static_kernel(const float2 *__restrict__ phi, int ns, int nkx, int nky,
                                                                double *__restrict__ scratch) {
  const int b = blockIdx.x;
  const bool row = b < nkx;
  const int fixed = row ? b : b - nkx;
  const int nfree = row ? nky : nkx;
  const long long slab = (long long)nkx * nky;
  double acc = 0.0;
  for (int q = threadIdx.x; q < ns * nfree; q += 256) {
    const int i = q / nfree, r = q - i * nfree;
    const int p = row ? fixed : r, m = row ? r : fixed;
    const float2 v = phi[(long long)i * slab + p * nky + m];
    const double a2 = (double)v.x * v.x + (double)v.y * v.y;
    acc += (m == 0 ? 1.0 : 2.0) * a2;
  }
  __shared__ double red[256];
  red[threadIdx.x] = acc;
  __syncthreads();
  for (int h = 128; h > 0; h >>= 1) {
    if (threadIdx.x < h) red[threadIdx.x] += red[threadIdx.x + h];
    __syncthreads();
  }
  if (threadIdx.x == 0) scratch[b] = red[0] / ns;
}

}  // namespace

extern "C" {

size_t gk_spectra_static_max(void) { return (size_t)kMaxOut; }

const char *gk_spectra_static_error(void) { return t_err; }

int gk_spectra_static(const void *phi_dev, int ns, int nkx, int nky, double *kx_spec_host, double *ky_spec_host,
                      void *cuda_stream) {
  t_err[0] = 0;
  // arguments first: nothing below touches the device until they are known to be good
  if (!phi_dev || !kx_spec_host || !ky_spec_host) return reject(GK_EINVAL, "gk_spectra_static: null pointer");
  if (ns < 1 || nkx < 1 || nky < 1) return reject(GK_EINVAL, "gk_spectra_static: ns, nkx, nky must be >= 1 (got %d, %d, %d)", ns, nkx, nky);
  if ((long long)nkx + nky > kMaxOut)
    return reject(GK_EINVAL, "gk_spectra_static: nkx + nky = %lld exceeds the fixed scratch of %d outputs "
                             "(GK_SPECTRA_STATIC_MAX); use gk_spectra with a context for larger planes",
                  (long long)nkx + nky, kMaxOut);
  if ((long long)ns * (nkx > nky ? nkx : nky) > 0x7fffffffLL)
    return reject(GK_EINVAL, "gk_spectra_static: ns * max(nkx, nky) does not fit 32-bit indexing");
  double *scratch = nullptr;
  if (int r = scratch_for_current_device(&scratch)) return r;
  cudaStream_t stream = (cudaStream_t)cuda_stream;
  const int n = nkx + nky;
  gk_spectra_static_kernel<<<n, 256, 0, stream>>>((const float2 *)phi_dev, ns, nkx, nky, scratch);
  cudaError_t e = cudaGetLastError();
  if (e == cudaSuccess) e = cudaMemcpyAsync(kx_spec_host, scratch, (size_t)nkx * sizeof(double), cudaMemcpyDeviceToHost, stream);
  if (e == cudaSuccess) e = cudaMemcpyAsync(ky_spec_host, scratch + nkx, (size_t)nky * sizeof(double), cudaMemcpyDeviceToHost, stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(stream);
  if (e != cudaSuccess) return reject(GK_ECUDA, "gk_spectra_static: %s", cudaGetErrorString(e));
  return GK_OK;
}

}  // extern "C"
