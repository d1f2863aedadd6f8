// hb_ws.cuh -- pieces shared by the warp-specialised persistent colour kernels (hb_sc_ws.cu, hb_bravais_ws.cu):
// the ring position, the tile scheduler's description, the round order of fused launches and their progress words.
#pragma once
#include "hb_device.cuh"
#include "hb_internal.h"

namespace hb {
namespace {

// position on a ring of N slots: slot index and the parity of the pass over the ring
template <int N>
struct RingPos {
  uint32_t slot = 0, par = 0;
  __device__ __forceinline__ void next() { if (++slot == N) { slot = 0; par ^= 1u; } }
};

struct WsTiles {
  int32_t n_ty, n_zc;   // tiles in y, chunks in z: chunk zc = planes [zc Lz / n_zc, (zc+1) Lz / n_zc), sizes differ by at most one
  uint32_t* sched;      // device, two words, zero between launches: next tile to hand out, CTAs that have finished
  // fused launches only: colour passes of the launch (pass p: sweep p / 2, colour p % 2), rounds between two passes (>= 3),
  // and passes x n_zc progress words, zero between launches: consumer warps that have finished a tile of (pass, k-th chunk)
  int32_t passes, lag;
  int32_t first;        // Bravais kernels: pass p updates colour (first + p) mod NB of sweep (first + p) / NB
  uint32_t* done;
  // diagnostic launches only (ALIAS, hb_probe_sc_l2): plane z is read and written at the address of plane z & zmask, so the
  // whole launch lives in a few L2-resident planes -- the kernel's rate with its HBM traffic taken away
  uint32_t zmask;
};

// a tile of a fused launch: pass, position k of its chunk in the pass's order, the chunk itself, the tile in y
struct FusedTile { int32_t p, k, zc, ty; };

// Round r holds the k-th chunk of pass p for r = lag p + k; within a round passes ascend.  S(r) = (pass, chunk) pairs in
// rounds before r = sum_p clamp(r - lag p, 0, n).
__device__ __forceinline__ FusedTile fused_decode(int32_t tile, const WsTiles& w) {
  const int32_t q = tile / w.n_ty, n = w.n_zc, P = w.passes, lag = w.lag;
  // passes 0 .. sat-1 have all n chunks behind them at round r, passes sat .. j-1 have r - lag p of them, the rest none
  auto before = [&](int32_t r) {
    const int32_t j = min(P, (r + lag - 1) / lag), sat = r >= n ? min(P, (r - n) / lag + 1) : 0;
    return sat * n + (j - sat) * r - lag * (((sat + j - 1) * (j - sat)) / 2);
  };
  int32_t lo = 0, hi = n + lag * (P - 1);   // before(lo) <= q < before(hi)
  while (hi - lo > 1) { const int32_t mid = (lo + hi) >> 1; if (before(mid) <= q) lo = mid; else hi = mid; }
  FusedTile t;
  t.p = (lo < n ? 0 : (lo - n) / lag + 1) + (q - before(lo));
  t.k = lo - lag * t.p;
  t.zc = (t.k + t.p) % n;
  t.ty = tile - q * w.n_ty;
  return t;
}

__device__ __forceinline__ uint32_t ld_acquire_gpu(const uint32_t* p) {
  uint32_t v;
  asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}

// the dynamic shared memory limit is an attribute of (function, device): set once per device
inline cudaError_t ws_configure(const void* kern, int bytes, unsigned long long& configured_mask) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 64 && ((configured_mask >> dev) & 1ull)) return cudaSuccess;
  e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
  if (e == cudaSuccess && dev < 64) configured_mask |= 1ull << dev;
  return e;
}

}  // namespace
}  // namespace hb
