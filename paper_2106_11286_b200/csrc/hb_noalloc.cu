// hb_noalloc.cu -- hb_measure_sc_noalloc (include/hb_noalloc.h): M and E of a simple cubic lattice for callers that
// must not allocate (all device memory owned by someone else's pool; a loop that cannot afford the device-wide stall of
// cudaMalloc / cudaFree; plug-in code that is handed input and output pointers and nothing more).
//
// It is the separate measurement pass of the library (k_measure_sc + k_reduce_final in hb_kernels.cu: per-site fp32
// terms, fp64 block partial sums, one block that adds the partials) rewritten for spins in canonical order and with
// the partial sums in the static array below instead of a context's workspace.  No existing path calls into this file
// and this file calls into none of them; it shares only the per-site energy term and the block reduction of
// hb_device.cuh.
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <mutex>

#include <cuda_runtime.h>

#include "../../include/hb.h"
#include "../../include/hb_noalloc.h"
#include "hb_device.cuh"

namespace {

using hb::block_reduce4;
using hb::site_energy;

constexpr int kThreads = 256;
constexpr int kSitesPerThread = HB_NOALLOC_SITES_PER_BLOCK / kThreads;   // 16
static_assert(kSitesPerThread * kThreads == HB_NOALLOC_SITES_PER_BLOCK, "a block's sites must divide among its threads");

// The scratch memory: 4 doubles (sum Sx, sum Sy, sum Sz, sum of the energy terms) per block of the first kernel.
// It is part of the library image, so every GPU that loads the image holds these 256 KiB until the process ends.
// In HOST code the name g_partials is only a handle for the runtime, not an address a kernel could use: the host
// function below turns it into this device's address with cudaGetSymbolAddress and hands that to the kernels.
// All calls on one GPU share it.  Nothing in it has to be zero: k_partial_sums writes entries [0, blocks) in full and
// k_total reads exactly those.
static __device__ __align__(256) double g_partials[HB_NOALLOC_MAX_BLOCKS * 4];
static_assert(sizeof(g_partials) == HB_NOALLOC_SCRATCH_BYTES, "the header states the size of the scratch array");

// Block b sums sites [4096 b, 4096 (b + 1)) of the canonical order; thread t takes sites t, t + 256, ... of that range
// (consecutive threads read consecutive floats).  Field and energy term exactly as the colour kernels form them
// (DESIGN.md 4.6): h = S(-x) + S(+x) + S(-y) + S(+y) + S(-z) + S(+z) in fp32, left to right.
__global__ void __launch_bounds__(kThreads)
k_partial_sums(const float* __restrict__ sx, const float* __restrict__ sy, const float* __restrict__ sz,
               uint32_t Lx, uint32_t Ly, uint32_t Lz, uint32_t n, float J, float K, float ex, float ey, float ez,
               double* partials) {
  const uint32_t plane = Lx * Ly;
  double mx = 0.0, my = 0.0, mz = 0.0, en = 0.0;
  const uint32_t first = blockIdx.x * (uint32_t)HB_NOALLOC_SITES_PER_BLOCK + threadIdx.x;
#pragma unroll 4
  for (int k = 0; k < kSitesPerThread; ++k) {
    const uint32_t i = first + (uint32_t)k * kThreads;
    if (i >= n) break;
    const uint32_t z = i / plane, r = i - z * plane, y = r / Lx, x = r - y * Lx;
    const uint32_t row = i - x;
    const uint32_t nb[6] = {
        row + (x == 0 ? Lx - 1 : x - 1), row + (x == Lx - 1 ? 0 : x + 1),
        y == 0 ? i + plane - Lx : i - Lx, y == Ly - 1 ? i - (plane - Lx) : i + Lx,
        z == 0 ? i + (n - plane) : i - plane, z == Lz - 1 ? i - (n - plane) : i + plane};
    float hx = __ldg(sx + nb[0]), hy = __ldg(sy + nb[0]), hz = __ldg(sz + nb[0]);
#pragma unroll
    for (int q = 1; q < 6; ++q) {
      hx = __fadd_rn(hx, __ldg(sx + nb[q]));
      hy = __fadd_rn(hy, __ldg(sy + nb[q]));
      hz = __fadd_rn(hz, __ldg(sz + nb[q]));
    }
    const float ox = __ldg(sx + i), oy = __ldg(sy + i), oz = __ldg(sz + i);
    mx += (double)ox; my += (double)oy; mz += (double)oz;
    en += (double)site_energy(ox, oy, oz, hx, hy, hz, J, K, ex, ey, ez);
  }
  block_reduce4(mx, my, mz, en, partials + (size_t)blockIdx.x * 4);
}

// One block adds the partial sums of `blocks` blocks and writes (M, E).
__global__ void __launch_bounds__(kThreads) k_total(const double* partials, int blocks, double inv_n, double* out) {
  double a[4] = {0.0, 0.0, 0.0, 0.0};
  for (int b = threadIdx.x; b < blocks; b += kThreads)
    for (int q = 0; q < 4; ++q) a[q] += partials[(size_t)b * 4 + q];
  __shared__ double tot[4];
  block_reduce4(a[0], a[1], a[2], a[3], tot);
  __syncthreads();
  if (threadIdx.x < 3) out[threadIdx.x] = tot[threadIdx.x] * inv_n;
  if (threadIdx.x == 3) out[3] = tot[3];
}

// The device address of g_partials, looked up once per device (set-up; see the header: "First call on each device").
constexpr int kMaxDevices = 64;
std::mutex g_lookup_mutex;
double* g_partials_addr[kMaxDevices];   // zero-initialised: "not looked up yet"

int fail(int status, char* err, size_t err_len, const char* fmt, ...) __attribute__((format(printf, 4, 5)));
int fail(int status, char* err, size_t err_len, const char* fmt, ...) {
  if (err && err_len) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(err, err_len, fmt, ap);
    va_end(ap);
  }
  return status;
}

}  // namespace

extern "C" int hb_measure_sc_noalloc(const float* sx, const float* sy, const float* sz, int32_t Lx, int32_t Ly, int32_t Lz,
                                     float J, float K, const float e[3], double* out, void* cuda_stream,
                                     char* err, size_t err_len) {
  if (err && err_len) err[0] = '\0';
  if (!sx || !sy || !sz || !out || !e)
    return fail(HB_EINVAL, err, err_len, "hb_measure_sc_noalloc: sx, sy, sz, out (device) and e (host) must not be NULL");
  if (Lx < 1 || Ly < 1 || Lz < 1)
    return fail(HB_EINVAL, err, err_len, "hb_measure_sc_noalloc: Lx, Ly, Lz must be >= 1 (got %d x %d x %d)", Lx, Ly, Lz);
  // three factors below 2^31 can overflow int64: bound the partial products before trusting the whole one
  const int64_t cap = HB_NOALLOC_MAX_SITES;
  const int64_t n = ((int64_t)Lx * Ly <= cap) ? (int64_t)Lx * Ly * Lz : cap + 1;
  if (n > cap)
    return fail(HB_EINVAL, err, err_len,
                "hb_measure_sc_noalloc: a lattice of %d x %d x %d sites is beyond the %lld sites the library's static scratch "
                "array (%d bytes) has room for; use hb_create / hb_measure with caller-provided buffers instead",
                Lx, Ly, Lz, (long long)HB_NOALLOC_MAX_SITES, (int)HB_NOALLOC_SCRATCH_BYTES);
  const double e2 = (double)e[0] * e[0] + (double)e[1] * e[1] + (double)e[2] * e[2];
  if (!std::isfinite(J) || !std::isfinite(K) || !std::isfinite(e2) || std::fabs(e2 - 1.0) > 1e-5)
    return fail(HB_EINVAL, err, err_len, "hb_measure_sc_noalloc: J and K must be finite and e a unit vector");

  // set-up, once per device, with that device current: the device address behind the host-side name g_partials
  int dev = -1;
  cudaError_t ce = cudaGetDevice(&dev);
  if (ce != cudaSuccess)
    return fail(HB_ECUDA, err, err_len, "hb_measure_sc_noalloc: cudaGetDevice: %s", cudaGetErrorString(ce));
  if (dev < 0 || dev >= kMaxDevices)
    return fail(HB_EINVAL, err, err_len, "hb_measure_sc_noalloc: device ordinal %d is outside 0..%d", dev, kMaxDevices - 1);
  double* partials = nullptr;
  {
    std::lock_guard<std::mutex> lock(g_lookup_mutex);
    if (!g_partials_addr[dev]) {
      void* p = nullptr;
      ce = cudaGetSymbolAddress(&p, g_partials);
      if (ce != cudaSuccess || !p)
        return fail(HB_ECUDA, err, err_len, "hb_measure_sc_noalloc: cudaGetSymbolAddress on device %d: %s", dev,
                    cudaGetErrorString(ce));
      g_partials_addr[dev] = static_cast<double*>(p);
    }
    partials = g_partials_addr[dev];
  }

  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const int blocks = (int)((n + HB_NOALLOC_SITES_PER_BLOCK - 1) / HB_NOALLOC_SITES_PER_BLOCK);   // 1 .. HB_NOALLOC_MAX_BLOCKS
  k_partial_sums<<<blocks, kThreads, 0, st>>>(sx, sy, sz, (uint32_t)Lx, (uint32_t)Ly, (uint32_t)Lz, (uint32_t)n, J, K,
                                              e[0], e[1], e[2], partials);
  ce = cudaGetLastError();
  if (ce != cudaSuccess)
    return fail(HB_ECUDA, err, err_len, "hb_measure_sc_noalloc: launch of the partial sums: %s", cudaGetErrorString(ce));
  k_total<<<1, kThreads, 0, st>>>(partials, blocks, 1.0 / (double)n, out);
  ce = cudaGetLastError();
  if (ce != cudaSuccess)
    return fail(HB_ECUDA, err, err_len, "hb_measure_sc_noalloc: launch of the total: %s", cudaGetErrorString(ce));
  return HB_OK;
}
