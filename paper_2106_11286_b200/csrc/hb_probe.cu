// hb_probe.cu -- the arithmetic ceiling of the colour kernels, measured on the device the library runs on.
//
// hb_probe_alu runs the attempt arithmetic of hb_device.cuh (Philox4x32-10, proposal, the five dependent adds of the
// neighbour sum per component, delta-H, acceptance) on registers only: no global or shared memory traffic inside the
// loop.  Four attempts per thread and iteration as two packed pairs, exactly as the sc kernels issue them, 256-thread
// blocks, 4 blocks per SM.  The rate it returns is what the instruction mix of the arithmetic contract (DESIGN.md
// section 4) allows on this chip at the clock it holds: the "alu" roofline bench.py reports beside the HBM one
// (DESIGN.md section 7).
#include <cstring>
#include <new>

#include "../../include/hb.h"
#include "../../include/hb_diag.h"
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

// ---- hb_probe_pipe: issue rates of the instruction kinds the colour kernels are made of (profiles/r01_pipe_rates.md) -------
namespace hb {
namespace {

// 8 independent register chains per thread, 64 instructions of the probed kind(s) per loop trip, timed with the SM clock
template <int KIND>
__global__ void __launch_bounds__(256, 4) k_probe_pipe(unsigned long long* per_sm, uint32_t* sink, int trips, uint32_t seed) {
  uint32_t a[8], b[8];
  float f[8], g[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) { a[i] = seed + threadIdx.x * 8u + i; b[i] = a[i] * 2654435761u; f[i] = 1.0f + 1e-3f * i; g[i] = 0.5f + 1e-3f * i; }
  const float c1 = 1.0000001f, c0 = 1e-9f;
  __syncthreads();
  const long long t0 = clock64();
  for (int t = 0; t < trips; ++t) {
#pragma unroll
    for (int r = 0; r < 8; ++r) {
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        if (KIND == HB_PIPE_FFMA || KIND == HB_PIPE_FFMA_WIDE_LOP3)
          asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(f[i]) : "f"(c1), "f"(c0));
        if (KIND == HB_PIPE_FFMA2 || KIND == HB_PIPE_FFMA2_WIDE_LOP3) {
          unsigned long long p, q, s;
          asm volatile("mov.b64 %0, {%1, %2};" : "=l"(p) : "f"(f[i]), "f"(g[i]));
          asm volatile("mov.b64 %0, {%1, %1};" : "=l"(q) : "f"(c1));
          asm volatile("mov.b64 %0, {%1, %1};" : "=l"(s) : "f"(c0));
          asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(p) : "l"(q), "l"(s));
          asm volatile("mov.b64 {%0, %1}, %2;" : "=f"(f[i]), "=f"(g[i]) : "l"(p));
        }
        if (KIND == HB_PIPE_IMAD)
          asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(a[i]) : "r"(0xD2511F53u), "r"(b[i]));
        if (KIND == HB_PIPE_IMAD_WIDE || KIND == HB_PIPE_WIDE_LOP3 || KIND == HB_PIPE_FFMA_WIDE_LOP3 || KIND == HB_PIPE_FFMA2_WIDE_LOP3) {
          unsigned long long w;
          asm volatile("mul.wide.u32 %0, %1, %2;" : "=l"(w) : "r"(a[i]), "r"(0xD2511F53u));
          if (KIND == HB_PIPE_IMAD_WIDE) asm volatile("{ .reg .u32 lo, hi; mov.b64 {lo, hi}, %1; add.u32 %0, lo, hi; }" : "=r"(a[i]) : "l"(w));   // (an add rides along)
          else asm volatile("{ .reg .u32 lo, hi; mov.b64 {lo, hi}, %2; lop3.b32 %0, lo, hi, %1, 0x96; }" : "=r"(a[i]) : "r"(b[i]), "l"(w));       // a Philox half round
        }
        if (KIND == HB_PIPE_LOP3)
          asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a[i]) : "r"(b[i]), "r"(seed));
      }
    }
  }
  const long long t1 = clock64();
  uint32_t acc = 0;
#pragma unroll
  for (int i = 0; i < 8; ++i) acc ^= a[i] ^ __float_as_uint(f[i]) ^ __float_as_uint(g[i]);
  if (acc == 0x12345u) sink[0] = acc;   // keeps the chains alive
  if (threadIdx.x == 0) {   // per SM (the clock is the SM's own): warps that ran there, first start, last end
    uint32_t smid;
    asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
    atomicAdd(per_sm + 3 * smid, (unsigned long long)(blockDim.x >> 5));
    atomicMin(per_sm + 3 * smid + 1, (unsigned long long)t0);
    atomicMax(per_sm + 3 * smid + 2, (unsigned long long)t1);
  }
}

constexpr int kProbeSmMax = 1024;

__global__ void k_probe_pipe_reset(unsigned long long* per_sm) {
  for (int i = threadIdx.x; i < kProbeSmMax; i += blockDim.x) { per_sm[3 * i] = 0ull; per_sm[3 * i + 1] = ~0ull; per_sm[3 * i + 2] = 0ull; }
}

template <int KIND>
cudaError_t probe_pipe_go(cudaStream_t st, unsigned long long* per_sm, uint32_t* sink, int blocks, int trips) {
  k_probe_pipe<KIND><<<blocks, 256, 0, st>>>(per_sm, sink, 16, 1u);   // warm-up
  k_probe_pipe_reset<<<1, 256, 0, st>>>(per_sm);
  k_probe_pipe<KIND><<<blocks, 256, 0, st>>>(per_sm, sink, trips, 1u);
  return cudaGetLastError();
}

}  // namespace
}  // namespace hb

extern "C" int hb_probe_pipe(void* cuda_stream, int32_t kind, double* warp_instr_per_clk_per_sm) {
  if (!warp_instr_per_clk_per_sm || kind < 0 || kind > HB_PIPE_FFMA2_WIDE_LOP3) return HB_EINVAL;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms < 1) return HB_ECUDA;
  const int blocks = sms * 4, trips = 2000;       // one wave: 4 blocks of 8 warps on every SM
  unsigned long long* cycles = nullptr;
  uint32_t* sink = nullptr;
  if (cudaMalloc(&cycles, (size_t)hb::kProbeSmMax * 24) != cudaSuccess || cudaMalloc(&sink, 4) != cudaSuccess) { cudaFree(cycles); cudaGetLastError(); return HB_ENOMEM; }
  cudaError_t e = cudaSuccess;
  switch (kind) {
    case HB_PIPE_FFMA: e = hb::probe_pipe_go<HB_PIPE_FFMA>(st, cycles, sink, blocks, trips); break;
    case HB_PIPE_FFMA2: e = hb::probe_pipe_go<HB_PIPE_FFMA2>(st, cycles, sink, blocks, trips); break;
    case HB_PIPE_IMAD: e = hb::probe_pipe_go<HB_PIPE_IMAD>(st, cycles, sink, blocks, trips); break;
    case HB_PIPE_IMAD_WIDE: e = hb::probe_pipe_go<HB_PIPE_IMAD_WIDE>(st, cycles, sink, blocks, trips); break;
    case HB_PIPE_LOP3: e = hb::probe_pipe_go<HB_PIPE_LOP3>(st, cycles, sink, blocks, trips); break;
    case HB_PIPE_WIDE_LOP3: e = hb::probe_pipe_go<HB_PIPE_WIDE_LOP3>(st, cycles, sink, blocks, trips); break;
    case HB_PIPE_FFMA_WIDE_LOP3: e = hb::probe_pipe_go<HB_PIPE_FFMA_WIDE_LOP3>(st, cycles, sink, blocks, trips); break;
    default: e = hb::probe_pipe_go<HB_PIPE_FFMA2_WIDE_LOP3>(st, cycles, sink, blocks, trips); break;
  }
  int rc = HB_ECUDA;
  if (e == cudaSuccess && cudaStreamSynchronize(st) == cudaSuccess) {
    unsigned long long* h = new (std::nothrow) unsigned long long[3 * hb::kProbeSmMax];
    if (h && cudaMemcpy(h, cycles, (size_t)hb::kProbeSmMax * 24, cudaMemcpyDeviceToHost) == cudaSuccess) {
      // probed instructions per warp and trip: 64 of each kind in the mix (the packing moves and adds that ride along are not counted)
      const int kinds_in_mix = kind == HB_PIPE_WIDE_LOP3 ? 2 : ((kind == HB_PIPE_FFMA_WIDE_LOP3 || kind == HB_PIPE_FFMA2_WIDE_LOP3) ? 3 : 1);
      const double per_warp = 64.0 * kinds_in_mix * trips;
      double sum = 0.0;
      int used = 0;
      for (int i = 0; i < hb::kProbeSmMax; ++i)       // every SM that ran warps: their instructions over its busy span
        if (h[3 * i] > 0 && h[3 * i + 2] > h[3 * i + 1]) { sum += (double)h[3 * i] * per_warp / (double)(h[3 * i + 2] - h[3 * i + 1]); used += 1; }
      if (used > 0) { *warp_instr_per_clk_per_sm = sum / used; rc = HB_OK; }
    }
    delete[] h;
  }
  cudaFree(cycles); cudaFree(sink);
  cudaGetLastError();
  return rc;
}

// ---- hb_device_math: the building blocks of an attempt, element by element (include/hb.h) ----------------------------------
namespace hb {
namespace {

// one thread per PAIR of elements (2t, 2t+1): the scalar path on each, and the packed fp32x2 path on the pair
__global__ void __launch_bounds__(256) k_device_math(int op, long long count, const uint32_t* in0, const uint32_t* in1, float* out) {
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const long long i = 2 * t, j = (i + 1 < count) ? i + 1 : i;
  if (i >= count) return;
  const uint32_t a0 = in0[i], b0 = in0[j];
  const uint32_t a1 = in1 ? in1[i] : 0u, b1 = in1 ? in1[j] : 0u;
  switch (op) {
    case HB_MATH_U01: {
      const f2 p = u01_2(a0, b0);
      out[2 * i] = u01(a0); out[2 * i + 1] = p.x;
      if (j != i) { out[2 * j] = u01(b0); out[2 * j + 1] = p.y; }
      break;
    }
    case HB_MATH_SINCOS: {   // scalar only: the packed evaluation is part of HB_MATH_SPHERE
      float s, c;
      sincos_spec((a0 >> 8) | 1u, s, c); out[2 * i] = s; out[2 * i + 1] = c;
      if (j != i) { sincos_spec((b0 >> 8) | 1u, s, c); out[2 * j] = s; out[2 * j + 1] = c; }
      break;
    }
    case HB_MATH_SPHERE: {
      float x, y, z;
      f2 nx, ny, nz;
      proposal2(Rand4{a0, a1, 0u, 0u}, Rand4{b0, b1, 0u, 0u}, nx, ny, nz);
      sphere(a0, a1, x, y, z);
      out[6 * i] = x; out[6 * i + 1] = y; out[6 * i + 2] = z; out[6 * i + 3] = nx.x; out[6 * i + 4] = ny.x; out[6 * i + 5] = nz.x;
      if (j != i) {
        sphere(b0, b1, x, y, z);
        out[6 * j] = x; out[6 * j + 1] = y; out[6 * j + 2] = z; out[6 * j + 3] = nx.y; out[6 * j + 4] = ny.y; out[6 * j + 5] = nz.y;
      }
      break;
    }
    case HB_MATH_EXP: {
      const f2 p = exp_spec2(make_float2(__uint_as_float(a0), __uint_as_float(b0)));
      out[2 * i] = exp_spec(__uint_as_float(a0)); out[2 * i + 1] = p.x;
      if (j != i) { out[2 * j] = exp_spec(__uint_as_float(b0)); out[2 * j + 1] = p.y; }
      break;
    }
    case HB_MATH_SQRT: {   // w = 1 - z^2 of the proposal from random word r0: sqrt_rn_unit(w) beside the IEEE square root
      const float za = __fmaf_rn(-2.0f, u01(a0), 1.0f), zb = __fmaf_rn(-2.0f, u01(b0), 1.0f);
      const float wa = __fmaf_rn(-za, za, 1.0f), wb = __fmaf_rn(-zb, zb, 1.0f);
      out[2 * i] = sqrt_rn_unit(wa); out[2 * i + 1] = __fsqrt_rn(wa);
      if (j != i) { out[2 * j] = sqrt_rn_unit(wb); out[2 * j + 1] = __fsqrt_rn(wb); }
      break;
    }
    case HB_MATH_ATTEMPT: {  // whole packed attempts against given old spins and fields: in0 = site ids, in1 = 16 words per
      // element (sweep_lo, sweep_hi, seed_lo, seed_hi, J, K, beta, ex, ey, ez, hx, hy, hz, sx, sy, sz as float bits)
      const uint32_t* pa = in1 + 16 * i; const uint32_t* pb = in1 + 16 * j;
      auto F = [](uint32_t w) { return __uint_as_float(w); };
      const Rand4 ra = philox4x32_10(a0, 0u, pa[0], pa[1], pa[2], pa[3]);
      const Rand4 rb = philox4x32_10(b0, 0u, pb[0], pb[1], pb[2], pb[3]);
      // the pair shares (J, K, beta, e) of element i, as the lanes of a kernel do
      f2 sx = make_float2(F(pa[13]), F(pb[13])), sy = make_float2(F(pa[14]), F(pb[14])), sz = make_float2(F(pa[15]), F(pb[15]));
      bool aa, ab;
      attempt2<ANISO_GENERAL>(ra, rb, F(pa[4]), F(pa[5]), F(pa[6]), F(pa[7]), F(pa[8]), F(pa[9]), make_float2(F(pa[10]), F(pb[10])),
                              make_float2(F(pa[11]), F(pb[11])), make_float2(F(pa[12]), F(pb[12])), sx, sy, sz, aa, ab);
      out[4 * i] = sx.x; out[4 * i + 1] = sy.x; out[4 * i + 2] = sz.x; out[4 * i + 3] = aa ? 1.0f : 0.0f;
      if (j != i) { out[4 * j] = sx.y; out[4 * j + 1] = sy.y; out[4 * j + 2] = sz.y; out[4 * j + 3] = ab ? 1.0f : 0.0f; }
      break;
    }
    default: break;
  }
}

}  // namespace
}  // namespace hb

extern "C" int hb_device_math(int32_t op, int64_t count, const uint32_t* in0, const uint32_t* in1, float* out) {
  static const int per_out[] = {2, 2, 6, 2, 2, 4};
  static const int per_in1[] = {0, 0, 1, 0, 0, 16};
  if (op < 0 || op > HB_MATH_ATTEMPT || count < 0 || count > (int64_t(1) << 26) || !in0 || !out || (per_in1[op] && !in1)) return HB_EINVAL;
  if (count == 0) return HB_OK;
  const size_t nb0 = (size_t)count * 4, nb1 = (size_t)count * 4 * per_in1[op], nbo = (size_t)count * 4 * per_out[op];
  uint32_t *d0 = nullptr, *d1 = nullptr;
  float* dout = nullptr;
  int rc = HB_OK;
  if (cudaMalloc(&d0, nb0) != cudaSuccess || (nb1 && cudaMalloc(&d1, nb1) != cudaSuccess) || cudaMalloc(&dout, nbo) != cudaSuccess) rc = HB_ENOMEM;
  if (rc == HB_OK) {
    cudaError_t e = cudaMemcpy(d0, in0, nb0, cudaMemcpyHostToDevice);
    if (e == cudaSuccess && nb1) e = cudaMemcpy(d1, in1, nb1, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) {
      const long long pairs = (count + 1) / 2;
      hb::k_device_math<<<(unsigned)((pairs + 255) / 256), 256>>>(op, (long long)count, d0, d1, dout);
      e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaMemcpy(out, dout, nbo, cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) rc = HB_ECUDA;
  }
  cudaFree(d0); cudaFree(d1); cudaFree(dout);
  cudaGetLastError();
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
