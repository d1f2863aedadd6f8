// hb_ell.cu -- colour kernels for arbitrary neighbour tables (free-surface nanostructures, per-site
// anisotropy) on the colour-major ELL layout of hb_internal.h.
//
// The spin state of this engine is AoS, one float4 (x, y, z, 0) per site in internal order: a neighbour
// is ONE 16-byte gather instead of three 4-byte ones from three planes, a third of the sector requests
// (the SoA planes of the structured kernels are for streaming, this path is gather-dominated).
// One thread per site of the colour.  Everything a warp streams is contiguous: its own spins, the
// per-site (K, e), the Philox site ids and, for each neighbour slot k, one word of the table per thread.
// Only the neighbour spins are gathered; they belong to other colours, whose sites are stored in
// canonical order inside their segment, so neighbouring threads gather neighbouring addresses and the
// gathers are served by L1/L2 (the whole spin state of config 5 is 43 MB).  The neighbour sum runs over
// the slots in order and skips the empty ones, which is the oracle's "for j in nn(i): h += S_j".
//
// HBM bytes per attempted update: table 4*maxdeg + site id 4 + (K, e) 16 + own
// spins 16 read + 16 written; neighbour spins once per colour pass at most.
#include "hb_device.cuh"
#include "hb_internal.h"

namespace hb {

namespace {

// neighbour field of the t-th site of a colour segment; MD > 0 unrolls the slot loop completely
template <int MD>
__device__ __forceinline__ void ell_field(const float4* __restrict__ S, const int32_t* __restrict__ e,
                                          uint32_t count, uint32_t maxdeg, float& hx, float& hy, float& hz) {
  hx = 0.0f; hy = 0.0f; hz = 0.0f;
  if constexpr (MD > 0) {
    int32_t j[MD];
#pragma unroll
    for (int k = 0; k < MD; ++k) j[k] = __ldcs(e + (size_t)k * count);   // streamed once per pass: evict first, keep L2 for spins
    float4 v[MD];
#pragma unroll
    for (int k = 0; k < MD; ++k) v[k] = __ldg(S + (j[k] < 0 ? 0 : j[k]));   // other colours: not written by this launch
#pragma unroll
    for (int k = 0; k < MD; ++k)
      if (j[k] >= 0) { hx = __fadd_rn(hx, v[k].x); hy = __fadd_rn(hy, v[k].y); hz = __fadd_rn(hz, v[k].z); }
  } else {
#pragma unroll 4
    for (uint32_t k = 0; k < maxdeg; ++k) {
      const int32_t q = __ldcs(e + (size_t)k * count);
      if (q >= 0) {
        const float4 v = __ldg(S + q);
        hx = __fadd_rn(hx, v.x); hy = __fadd_rn(hy, v.y); hz = __fadd_rn(hz, v.z);
      }
    }
  }
}

template <int MD, bool DIAG>
__global__ void __launch_bounds__(256)
k_sweep_ell(float4* S, EllDev g, uint32_t begin, uint32_t count, SweepParams P, Diag d) {
  resolve_sweep(P);
  const uint32_t t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= count) return;
  const uint32_t m = begin + t;
  const int32_t* e = g.ell + (size_t)g.maxdeg * begin + t;
  float hx = 0.0f, hy = 0.0f, hz = 0.0f;
  float K = P.K, ex = P.ex, ey = P.ey, ez = P.ez;
  uint32_t site;
  float4 o;
  if constexpr (MD > 0) {
    // everything that does not depend on another load (table words, site id, anisotropy, own spin) is requested before
    // the gathers: the kernel is a chain of memory latencies, not of arithmetic (c5: 26.9 -> 28.4 Gupd/s greedy, 41 -> 43.8
    // parity).  Forcing all gathers of a site into flight at once (__launch_bounds__(256, 3), 80 registers) gives 29.5 /
    // 40.9: what the greedy colouring gains in latency the balanced one loses in occupancy, so the bound stays open.
    int32_t j[MD];
#pragma unroll
    for (int k = 0; k < MD; ++k) j[k] = __ldcs(e + (size_t)k * count);   // streamed once per pass: evict first, keep L2 for spins
    site = (uint32_t)__ldcs(g.perm + m);
    if (g.K) { K = __ldcs(g.K + m); ex = __ldcs(g.ex + m); ey = __ldcs(g.ey + m); ez = __ldcs(g.ez + m); }
    o = S[m];
    float4 v[MD];
#pragma unroll
    for (int k = 0; k < MD; ++k) v[k] = __ldg(S + (j[k] < 0 ? 0 : j[k]));   // other colours: not written by this launch
#pragma unroll
    for (int k = 0; k < MD; ++k)
      if (j[k] >= 0) { hx = __fadd_rn(hx, v[k].x); hy = __fadd_rn(hy, v[k].y); hz = __fadd_rn(hz, v[k].z); }
  } else {
    ell_field<MD>(S, e, count, g.maxdeg, hx, hy, hz);
    if (g.K) { K = __ldcs(g.K + m); ex = __ldcs(g.ex + m); ey = __ldcs(g.ey + m); ez = __ldcs(g.ez + m); }
    site = (uint32_t)__ldcs(g.perm + m);
    o = S[m];
  }
  const Rand4 r = philox4x32_10(site + g.site_base, 0u, P.sweep_lo, P.sweep_hi, P.seed_lo, P.seed_hi);
  float nx, ny, nz;
  sphere(r.r0, r.r1, nx, ny, nz);
  const float dH = delta_h(o.x, o.y, o.z, nx, ny, nz, hx, hy, hz, P.J, K, ex, ey, ez);
  const bool acc = metropolis_accept(dH, P.beta, r.r2);
  if (acc) S[m] = make_float4(nx, ny, nz, 0.0f);
  if (DIAG) {
    if (d.accept) d.accept[site] = acc;
    if (d.n_accept) {   // one atomic per warp (some lanes of the last warp have left)
      const unsigned live = __activemask(), votes = __ballot_sync(live, acc);
      if (votes && (threadIdx.x & 31) == (unsigned)(__ffs(live) - 1)) atomicAdd(d.n_accept, (unsigned long long)__popc(votes));
    }
  }
}

template <int MD>
__global__ void __launch_bounds__(256)
k_measure_ell(const float4* __restrict__ S, EllDev g, SweepParams P, double* partials) {
  double mx = 0, my = 0, mz = 0, en = 0;
  for (int c = 0; c < g.n_colours; ++c) {
    const uint32_t begin = g.colour_begin[c], count = g.colour_begin[c + 1] - begin;
    for (uint32_t t = blockIdx.x * blockDim.x + threadIdx.x; t < count; t += gridDim.x * blockDim.x) {
      const uint32_t m = begin + t;
      float hx, hy, hz;
      ell_field<MD>(S, g.ell + (size_t)g.maxdeg * begin + t, count, g.maxdeg, hx, hy, hz);
      float K = P.K, ex = P.ex, ey = P.ey, ez = P.ez;
      if (g.K) { K = __ldg(g.K + m); ex = __ldg(g.ex + m); ey = __ldg(g.ey + m); ez = __ldg(g.ez + m); }
      const float4 o = __ldg(S + m);
      mx += (double)o.x; my += (double)o.y; mz += (double)o.z;
      en += (double)site_energy(o.x, o.y, o.z, hx, hy, hz, P.J, K, ex, ey, ez);
    }
  }
  block_reduce4(mx, my, mz, en, partials + (size_t)blockIdx.x * 4);
}

__global__ void k_init_random_perm(float4* S, const int32_t* __restrict__ perm, uint32_t n, uint32_t seed_lo, uint32_t seed_hi, uint32_t site_base) {
  for (unsigned long long m64 = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; m64 < n; m64 += (unsigned long long)gridDim.x * blockDim.x) {
    const uint32_t m = (uint32_t)m64;   // 64-bit loop index: a 32-bit one wraps below n when n is close to 2^32
    const Rand4 r = philox4x32_10((uint32_t)perm[m] + site_base, 1u, 0u, 0u, seed_lo, seed_hi);
    float x, y, z;
    sphere(r.r0, r.r1, x, y, z);
    S[m] = make_float4(x, y, z, 0.0f);
  }
}

__global__ void k_fill4(float4* S, uint32_t n, float x, float y, float z) {
  for (unsigned long long m = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; m < n; m += (unsigned long long)gridDim.x * blockDim.x) S[m] = make_float4(x, y, z, 0.0f);
}

// component comp of the internal AoS state <-> one canonical plane
__global__ void k_permute(float4* S, float* plane, const int32_t* __restrict__ perm, uint32_t n, int comp, bool to_internal) {
  float* s = reinterpret_cast<float*>(S);
  for (unsigned long long m64 = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; m64 < n; m64 += (unsigned long long)gridDim.x * blockDim.x) {
    const uint32_t m = (uint32_t)m64;   // 64-bit loop index: a 32-bit one wraps below n when n is close to 2^32
    if (to_internal) s[4 * (size_t)m + comp] = plane[perm[m]]; else plane[perm[m]] = s[4 * (size_t)m + comp];
  }
}

// exchange step of table parts: the spins of the listed local sites <-> packed (x, y, z, 0) records
__global__ void k_part_move_ell(float4* S, const int32_t* __restrict__ inv, const int32_t* __restrict__ ids, uint32_t count, float4* packed, bool gather) {
  for (unsigned long long k = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; k < count; k += (unsigned long long)gridDim.x * blockDim.x) {
    const int32_t m = inv[ids[k]];
    if (gather) packed[k] = S[m]; else { const float4 v = packed[k]; S[m] = make_float4(v.x, v.y, v.z, 0.0f); }
  }
}

inline int grid_cap(uint32_t n, int block, int cap) {
  const long long g = ((long long)n + block - 1) / block;
  return (int)(g < 1 ? 1 : (g > cap ? cap : g));
}

template <int MD>
cudaError_t sweep_go(cudaStream_t st, float* s, const EllDev& g, uint32_t begin, uint32_t count, const SweepParams& p,
                     int block, const Diag& d) {
  float4* S = reinterpret_cast<float4*>(s);
  const int grid = (int)((count + block - 1) / block);
  if (d.accept || d.n_accept) return launch_colour_kernel(k_sweep_ell<MD, true>, dim3(grid), dim3(block), 0, st, p.pdl != 0, S, g, begin, count, p, d);
  return launch_colour_kernel(k_sweep_ell<MD, false>, dim3(grid), dim3(block), 0, st, p.pdl != 0, S, g, begin, count, p, d);
}

}  // namespace

cudaError_t launch_sweep_ell(cudaStream_t st, float* s, EllDev g, uint32_t begin, uint32_t count, SweepParams p,
                             int block, Diag d) {
  if (count == 0) return cudaSuccess;
  switch (g.maxdeg) {   // the coordination numbers of the paper's lattices get fully unrolled slot loops
    case 6: return sweep_go<6>(st, s, g, begin, count, p, block, d);
    case 8: return sweep_go<8>(st, s, g, begin, count, p, block, d);
    case 12: return sweep_go<12>(st, s, g, begin, count, p, block, d);
    default: return sweep_go<0>(st, s, g, begin, count, p, block, d);
  }
}

cudaError_t launch_measure_ell(cudaStream_t st, const float* s, EllDev g, SweepParams p, double* partials, double* out) {
  const float4* S = reinterpret_cast<const float4*>(s);
  const int grid = grid_cap(g.n / (g.n_colours > 0 ? g.n_colours : 1) + 1, 256, kMeasureBlocks);
  switch (g.maxdeg) {
    case 6: k_measure_ell<6><<<grid, 256, 0, st>>>(S, g, p, partials); break;
    case 8: k_measure_ell<8><<<grid, 256, 0, st>>>(S, g, p, partials); break;
    case 12: k_measure_ell<12><<<grid, 256, 0, st>>>(S, g, p, partials); break;
    default: k_measure_ell<0><<<grid, 256, 0, st>>>(S, g, p, partials); break;
  }
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  return launch_reduce_final(st, partials, grid, out);
}

cudaError_t launch_init_random_perm(cudaStream_t st, float* s, const int32_t* perm, uint32_t n, uint32_t seed_lo, uint32_t seed_hi, uint32_t site_base) {
  k_init_random_perm<<<grid_cap(n, 256, 148 * 16), 256, 0, st>>>(reinterpret_cast<float4*>(s), perm, n, seed_lo, seed_hi, site_base);
  return cudaGetLastError();
}

cudaError_t launch_part_move_ell(cudaStream_t st, float* s, const int32_t* inv, const int32_t* ids, uint32_t count, float* packed, bool gather) {
  if (count == 0) return cudaSuccess;
  k_part_move_ell<<<grid_cap(count, 256, 148 * 8), 256, 0, st>>>(reinterpret_cast<float4*>(s), inv, ids, count, reinterpret_cast<float4*>(packed), gather);
  return cudaGetLastError();
}

cudaError_t launch_fill_ell(cudaStream_t st, float* s, uint32_t n, float x, float y, float z) {
  k_fill4<<<grid_cap(n, 256, 148 * 16), 256, 0, st>>>(reinterpret_cast<float4*>(s), n, x, y, z);
  return cudaGetLastError();
}

cudaError_t launch_permute_ell(cudaStream_t st, float* s, float* plane, const int32_t* perm, uint32_t n, int comp, bool to_internal) {
  k_permute<<<grid_cap(n, 256, 148 * 16), 256, 0, st>>>(reinterpret_cast<float4*>(s), plane, perm, n, comp, to_internal);
  return cudaGetLastError();
}

}  // namespace hb
