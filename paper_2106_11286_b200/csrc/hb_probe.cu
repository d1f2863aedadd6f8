// hb_probe.cu -- the arithmetic ceiling of the colour kernels, measured on the device the library runs on.
//
// hb_probe_alu runs the attempt arithmetic of hb_device.cuh (Philox4x32-10, proposal, the five dependent adds of the
// neighbour sum per component, delta-H, acceptance) on registers only: no global or shared memory traffic inside the
// loop.  Four attempts per thread and iteration as two packed pairs, exactly as the sc kernels issue them, 256-thread
// blocks, 4 blocks per SM.  The rate it returns is what the instruction mix of the arithmetic contract (DESIGN.md
// section 4) allows on this chip at the clock it holds: the "alu" roofline bench.py reports beside the HBM one
// (DESIGN.md section 7).
#include <cstring>

#include "../../include/hb.h"
#include "hb_device.cuh"
#include "hb_internal.h"

namespace hb {
namespace {

__global__ void __launch_bounds__(256, 4) k_probe_alu(float* out, int n_iter, uint32_t seed, float beta, float K) {
  const uint32_t site = (blockIdx.x * blockDim.x + threadIdx.x) * 8u;
  f2 sx0 = make_float2(0.0f, 0.6f), sy0 = make_float2(0.0f, 0.8f), sz0 = make_float2(1.0f, 0.0f);
  f2 sx1 = sx0, sy1 = sy0, sz1 = sz0;
  const f2 hx = make_float2(0.5f, -0.3f), hy = make_float2(1.5f, 0.3f), hz = make_float2(-2.5f, 0.1f);
  for (int it = 0; it < n_iter; ++it) {
    const Rand4 ra = philox4x32_10(site, 0u, (uint32_t)it, 0u, seed, 7u);
    const Rand4 rb = philox4x32_10(site + 2u, 0u, (uint32_t)it, 0u, seed, 7u);
    const Rand4 rc = philox4x32_10(site + 4u, 0u, (uint32_t)it, 0u, seed, 7u);
    const Rand4 rd = philox4x32_10(site + 6u, 0u, (uint32_t)it, 0u, seed, 7u);
    f2 gx = hx, gy = hy, gz = hz, kx = hx, ky = hy, kz = hz;
#pragma unroll
    for (int q = 0; q < 5; ++q) {   // the neighbour sum: five dependent adds per component and pair
      gx = add2(gx, sx1); gy = add2(gy, sy1); gz = add2(gz, sz1);
      kx = add2(kx, sx0); ky = add2(ky, sy0); kz = add2(kz, sz0);
    }
    bool a, b, c, d;
    attempt2<ANISO_Z>(ra, rb, 1.0f, K, beta, 0.0f, 0.0f, 1.0f, gx, gy, gz, sx0, sy0, sz0, a, b);
    attempt2<ANISO_Z>(rc, rd, 1.0f, K, beta, 0.0f, 0.0f, 1.0f, kx, ky, kz, sx1, sy1, sz1, c, d);
  }
  out[blockIdx.x * blockDim.x + threadIdx.x] =
      sx0.x + sx0.y + sy0.x + sy0.y + sz0.x + sz0.y + sx1.x + sx1.y + sy1.x + sy1.y + sz1.x + sz1.y;
}

}  // namespace
}  // namespace hb

extern "C" int hb_probe_alu(void* cuda_stream, double seconds, double* updates_per_second) {
  if (!updates_per_second || !(seconds > 0.0) || seconds > 10.0) return HB_EINVAL;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms < 1)
    return HB_ECUDA;
  const int blocks = sms * 4 * 4, threads = 256, n_iter = 200;
  float* out = nullptr;
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  if (cudaMalloc(&out, (size_t)blocks * threads * sizeof(float)) != cudaSuccess) return HB_ENOMEM;
  int rc = HB_ECUDA;
  if (cudaEventCreate(&e0) == cudaSuccess && cudaEventCreate(&e1) == cudaSuccess) {
    // launches back to back for about `seconds`, so that the clock is the one a long run holds; the last half is timed
    const double per_launch = (double)blocks * threads * 4.0 * n_iter;
    hb::k_probe_alu<<<blocks, threads, 0, st>>>(out, n_iter, 1u, 0.7f, 0.01f);
    cudaEventRecord(e0, st);
    hb::k_probe_alu<<<blocks, threads, 0, st>>>(out, n_iter, 1u, 0.7f, 0.01f);
    cudaEventRecord(e1, st);
    float ms = 0.0f;
    if (cudaEventSynchronize(e1) == cudaSuccess && cudaEventElapsedTime(&ms, e0, e1) == cudaSuccess && ms > 0.0f) {
      const int n_launch = (int)(seconds * 1e3 / ms / 2.0) + 1;
      for (int i = 0; i < n_launch; ++i) hb::k_probe_alu<<<blocks, threads, 0, st>>>(out, n_iter, 1u, 0.7f, 0.01f);
      cudaEventRecord(e0, st);
      for (int i = 0; i < n_launch; ++i) hb::k_probe_alu<<<blocks, threads, 0, st>>>(out, n_iter, 1u, 0.7f, 0.01f);
      cudaEventRecord(e1, st);
      if (cudaEventSynchronize(e1) == cudaSuccess && cudaEventElapsedTime(&ms, e0, e1) == cudaSuccess && ms > 0.0f &&
          cudaGetLastError() == cudaSuccess) {
        *updates_per_second = per_launch * n_launch / (ms * 1e-3);
        rc = HB_OK;
      }
    }
  }
  if (e0) cudaEventDestroy(e0);
  if (e1) cudaEventDestroy(e1);
  cudaFree(out);
  return rc;
}

// ---- device memory another process can map (include/hb.h) ----------------------------------------------------------------
static_assert(sizeof(cudaIpcMemHandle_t) == 64, "CUDA IPC handle size");

extern "C" int hb_device_alloc(size_t bytes, void** ptr) {
  if (!ptr || bytes == 0) return HB_EINVAL;
  *ptr = nullptr;
  const cudaError_t e = cudaMalloc(ptr, bytes);
  if (e != cudaSuccess) { cudaGetLastError(); return e == cudaErrorMemoryAllocation ? HB_ENOMEM : HB_ECUDA; }
  return HB_OK;
}

extern "C" int hb_device_free(void* ptr) {
  if (!ptr) return HB_OK;
  return cudaFree(ptr) == cudaSuccess ? HB_OK : HB_ECUDA;
}

extern "C" int hb_ipc_export(void* ptr, unsigned char handle[64]) {
  if (!ptr || !handle) return HB_EINVAL;
  cudaIpcMemHandle_t h;
  if (cudaIpcGetMemHandle(&h, ptr) != cudaSuccess) { cudaGetLastError(); return HB_ECUDA; }
  memcpy(handle, &h, sizeof h);
  return HB_OK;
}

extern "C" int hb_ipc_open(const unsigned char handle[64], void** ptr) {
  if (!handle || !ptr) return HB_EINVAL;
  cudaIpcMemHandle_t h;
  memcpy(&h, handle, sizeof h);
  *ptr = nullptr;
  if (cudaIpcOpenMemHandle(ptr, h, cudaIpcMemLazyEnablePeerAccess) != cudaSuccess) { cudaGetLastError(); return HB_ECUDA; }
  return HB_OK;
}

extern "C" int hb_ipc_close(void* ptr) {
  if (!ptr) return HB_OK;
  return cudaIpcCloseMemHandle(ptr) == cudaSuccess ? HB_OK : HB_ECUDA;
}
