// hb_kernels.cu -- sm_100a kernels of the Metropolis colour sweep.
//
//   k_sweep_sc    one colour of the simple-cubic checkerboard, colour-split SoA planes,
//                 128-bit loads/stores, a block owns an (x-chunk, y-tile) column and marches z
//   k_sweep_csr   one colour of an arbitrary neighbour table (free-boundary nanostructures)
//   k_measure_*   M (eq. 2) and E (eq. 1): warp shuffles, block partials, fixed-order final sum
//   k_init_*      initial states, layout permutation for host set/get
//
// No tensor cores: the path is not a contraction.  HBM traffic per attempted update is
// the roofline quantity (36 B for two colours); see DESIGN.md section 7.
#include "hb_device.cuh"
#include "hb_internal.h"

namespace hb {

namespace {

// ---- small vector helpers: V consecutive floats ------------------------------------------
template <int V> struct Vec { float v[V]; };

template <int V> __device__ __forceinline__ Vec<V> load_ro(const float* p);   // read-only path
template <> __device__ __forceinline__ Vec<4> load_ro<4>(const float* p) {
  const float4 t = __ldg(reinterpret_cast<const float4*>(p));
  return Vec<4>{{t.x, t.y, t.z, t.w}};
}
template <> __device__ __forceinline__ Vec<2> load_ro<2>(const float* p) {
  const float2 t = __ldg(reinterpret_cast<const float2*>(p));
  return Vec<2>{{t.x, t.y}};
}
template <> __device__ __forceinline__ Vec<1> load_ro<1>(const float* p) { return Vec<1>{{__ldg(p)}}; }

template <int V> __device__ __forceinline__ Vec<V> load_rw(const float* p);
template <> __device__ __forceinline__ Vec<4> load_rw<4>(const float* p) {
  const float4 t = *reinterpret_cast<const float4*>(p);
  return Vec<4>{{t.x, t.y, t.z, t.w}};
}
template <> __device__ __forceinline__ Vec<2> load_rw<2>(const float* p) {
  const float2 t = *reinterpret_cast<const float2*>(p);
  return Vec<2>{{t.x, t.y}};
}
template <> __device__ __forceinline__ Vec<1> load_rw<1>(const float* p) { return Vec<1>{{*p}}; }

template <int V> __device__ __forceinline__ void store(float* p, const Vec<V>& a);
template <> __device__ __forceinline__ void store<4>(float* p, const Vec<4>& a) {
  *reinterpret_cast<float4*>(p) = make_float4(a.v[0], a.v[1], a.v[2], a.v[3]);
}
template <> __device__ __forceinline__ void store<2>(float* p, const Vec<2>& a) {
  *reinterpret_cast<float2*>(p) = make_float2(a.v[0], a.v[1]);
}
template <> __device__ __forceinline__ void store<1>(float* p, const Vec<1>& a) { *p = a.v[0]; }

// ---- simple cubic, colour-split layout -----------------------------------------------------
// Plane c of a component holds the sites with (x+y+z) mod 2 == c, row (y,z) of H = Lx/2 floats:
// element i of that row is x = 2 i + ((c+y+z) & 1).  For a site of colour c in row (y,z), with
// p = (c+y+z) & 1, the six neighbours live in the other colour's plane at
//   -x,+x : row (y,z), elements i-1+p and i+p        -y,+y : rows (y-1,z),(y+1,z), element i
//   -z,+z : rows (y,z-1),(y,z+1), element i                                 (all periodic)
//
// Neighbour field of the V sites [i0, i0+V) of row (y,z): h = S(-x)+S(+x)+S(-y)+S(+y)+S(-z)+S(+z),
// summed in that order (the two x terms commute bitwise).
template <int V>
__device__ __forceinline__ Vec<V> sc_field(const float* __restrict__ b, const ScLayout& L, uint32_t row_c,
                                           uint32_t row_ym, uint32_t row_yp, uint32_t row_zm, uint32_t row_zp,
                                           int32_t i0, int32_t p) {
  const Vec<V> c = load_ro<V>(b + row_c + i0);
  int32_t ih = p ? i0 + V : i0 - 1;                 // the one element outside [i0, i0+V)
  ih = ih < 0 ? ih + L.H : (ih >= L.H ? ih - L.H : ih);
  const float halo = __ldg(b + row_c + ih);
  const Vec<V> ym = load_ro<V>(b + row_ym + i0);
  const Vec<V> yp = load_ro<V>(b + row_yp + i0);
  const Vec<V> zm = load_ro<V>(b + row_zm + i0);
  const Vec<V> zp = load_ro<V>(b + row_zp + i0);
  Vec<V> h;
#pragma unroll
  for (int k = 0; k < V; ++k) {
    const float lo = (k == 0) ? halo : c.v[k > 0 ? k - 1 : 0];          // p = 0: elements i-1, i
    const float hi = (k == V - 1) ? halo : c.v[k < V - 1 ? k + 1 : 0];  // p = 1: elements i, i+1
    float s = __fadd_rn(c.v[k], p ? hi : lo);
    s = __fadd_rn(s, ym.v[k]);
    s = __fadd_rn(s, yp.v[k]);
    s = __fadd_rn(s, zm.v[k]);
    s = __fadd_rn(s, zp.v[k]);
    h.v[k] = s;
  }
  return h;
}

// one Metropolis attempt (steps ii-iii of the paper) on registers; returns the decision
__device__ __forceinline__ bool attempt(uint32_t site, const SweepParams& P, float K, float ex, float ey, float ez,
                                        float hx, float hy, float hz, float& sx, float& sy, float& sz) {
  const Rand4 r = philox4x32_10(site, 0u, P.sweep_lo, P.sweep_hi, P.seed_lo, P.seed_hi);
  float nx, ny, nz;
  sphere(r.r0, r.r1, nx, ny, nz);
  const float dH = delta_h(sx, sy, sz, nx, ny, nz, hx, hy, hz, P.J, K, ex, ey, ez);
  const bool acc = metropolis_accept(dH, P.beta, r.r2);
  sx = acc ? nx : sx;
  sy = acc ? ny : sy;
  sz = acc ? nz : sz;
  return acc;
}

template <int V, bool DIAG>
__global__ void __launch_bounds__(256)
k_sweep_sc(float* __restrict__ ax, float* __restrict__ ay, float* __restrict__ az,
           const float* __restrict__ bx, const float* __restrict__ by, const float* __restrict__ bz,
           ScLayout L, ScTile t, SweepParams P, int colour, Diag d) {
  const int32_t tj = threadIdx.x % t.JX, ty = threadIdx.x / t.JX;
  const int32_t j = blockIdx.x * t.JX + tj;
  const int32_t y = blockIdx.y * t.TY + ty;
  const int32_t i0 = j * V;
  if (i0 >= L.H || y >= L.Ly) return;
  const int32_t ym = (y == 0) ? L.Ly - 1 : y - 1;
  const int32_t yp = (y == L.Ly - 1) ? 0 : y + 1;
  const int32_t z0 = blockIdx.z * t.ZT;
  const int32_t z1 = min(z0 + t.ZT, L.Lz);
  unsigned n_acc = 0;
  for (int32_t z = z0; z < z1; ++z) {
    const int32_t zm = (z == 0) ? L.Lz - 1 : z - 1;
    const int32_t zp = (z == L.Lz - 1) ? 0 : z + 1;
    const int32_t p = (colour + y + z) & 1;
    const uint32_t row_c = (uint32_t)(z * L.Ly + y) * L.H;
    const uint32_t row_ym = (uint32_t)(z * L.Ly + ym) * L.H, row_yp = (uint32_t)(z * L.Ly + yp) * L.H;
    const uint32_t row_zm = (uint32_t)(zm * L.Ly + y) * L.H, row_zp = (uint32_t)(zp * L.Ly + y) * L.H;
    const Vec<V> hx = sc_field<V>(bx, L, row_c, row_ym, row_yp, row_zm, row_zp, i0, p);
    const Vec<V> hy = sc_field<V>(by, L, row_c, row_ym, row_yp, row_zm, row_zp, i0, p);
    const Vec<V> hz = sc_field<V>(bz, L, row_c, row_ym, row_yp, row_zm, row_zp, i0, p);
    Vec<V> sx = load_rw<V>(ax + row_c + i0), sy = load_rw<V>(ay + row_c + i0), sz = load_rw<V>(az + row_c + i0);
    const uint32_t site0 = (uint32_t)(z * L.Ly + y) * (uint32_t)L.Lx + 2u * (uint32_t)i0 + (uint32_t)p;
    bool any = false;
#pragma unroll
    for (int k = 0; k < V; ++k) {
      const bool acc = attempt(site0 + 2u * k, P, P.K, P.ex, P.ey, P.ez, hx.v[k], hy.v[k], hz.v[k],
                               sx.v[k], sy.v[k], sz.v[k]);
      any |= acc;
      if (DIAG) {
        n_acc += acc;
        if (d.accept) d.accept[site0 + 2u * k] = acc;
      }
    }
    if (any) {
      store<V>(ax + row_c + i0, sx);
      store<V>(ay + row_c + i0, sy);
      store<V>(az + row_c + i0, sz);
    }
  }
  if (DIAG && d.n_accept && n_acc) atomicAdd(d.n_accept, (unsigned long long)n_acc);
}

// ---- CSR: one thread per site of the colour -------------------------------------------------
template <bool DIAG>
__global__ void __launch_bounds__(256)
k_sweep_csr(float* sx, float* sy, float* sz, CsrDev g, uint32_t list_begin, uint32_t list_count,
            SweepParams P, Diag d) {
  const uint32_t t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= list_count) return;
  const uint32_t i = (uint32_t)g.list[list_begin + t];
  const int32_t k0 = g.row_ptr[i], k1 = g.row_ptr[i + 1];
  float hx = 0.0f, hy = 0.0f, hz = 0.0f;
  for (int32_t k = k0; k < k1; ++k) {
    const int32_t j = __ldg(g.col + k);
    hx = __fadd_rn(hx, sx[j]);
    hy = __fadd_rn(hy, sy[j]);
    hz = __fadd_rn(hz, sz[j]);
  }
  float K = P.K, ex = P.ex, ey = P.ey, ez = P.ez;
  if (g.K_site) {
    K = __ldg(g.K_site + i);
    ex = __ldg(g.e_site + 3 * (size_t)i);
    ey = __ldg(g.e_site + 3 * (size_t)i + 1);
    ez = __ldg(g.e_site + 3 * (size_t)i + 2);
  }
  float ox = sx[i], oy = sy[i], oz = sz[i];
  const bool acc = attempt(i, P, K, ex, ey, ez, hx, hy, hz, ox, oy, oz);
  if (acc) { sx[i] = ox; sy[i] = oy; sz[i] = oz; }
  if (DIAG) {
    if (d.accept) d.accept[i] = acc;
    if (d.n_accept && acc) atomicAdd(d.n_accept, 1ull);
  }
}

// ---- initial states -----------------------------------------------------------------------------
__device__ __forceinline__ uint32_t sc_canonical(const ScLayout& L, uint32_t m) {
  // internal index m = c*half + (z*Ly + y)*H + i  ->  canonical id (z*Ly + y)*Lx + 2i + ((c+y+z)&1)
  const uint32_t c = m >= L.half ? 1u : 0u;
  const uint32_t r = m - c * L.half;
  const uint32_t row = r / (uint32_t)L.H, i = r - row * (uint32_t)L.H;
  const uint32_t z = row / (uint32_t)L.Ly, y = row - z * (uint32_t)L.Ly;
  return row * (uint32_t)L.Lx + 2u * i + ((c + y + z) & 1u);
}

__global__ void k_init_random_sc(float* sx, float* sy, float* sz, ScLayout L, uint32_t seed_lo, uint32_t seed_hi) {
  for (uint32_t m = blockIdx.x * blockDim.x + threadIdx.x; m < L.n; m += gridDim.x * blockDim.x) {
    const Rand4 r = philox4x32_10(sc_canonical(L, m), 1u, 0u, 0u, seed_lo, seed_hi);
    float x, y, z;
    sphere(r.r0, r.r1, x, y, z);
    sx[m] = x; sy[m] = y; sz[m] = z;
  }
}

__global__ void k_init_random_flat(float* sx, float* sy, float* sz, uint32_t n, uint32_t seed_lo, uint32_t seed_hi) {
  for (uint32_t m = blockIdx.x * blockDim.x + threadIdx.x; m < n; m += gridDim.x * blockDim.x) {
    const Rand4 r = philox4x32_10(m, 1u, 0u, 0u, seed_lo, seed_hi);
    float x, y, z;
    sphere(r.r0, r.r1, x, y, z);
    sx[m] = x; sy[m] = y; sz[m] = z;
  }
}

__global__ void k_fill(float* sx, float* sy, float* sz, uint32_t n, float x, float y, float z) {
  for (uint32_t m = blockIdx.x * blockDim.x + threadIdx.x; m < n; m += gridDim.x * blockDim.x) {
    sx[m] = x; sy[m] = y; sz[m] = z;
  }
}

// dst[m] = src[canonical(m)] (to_internal) or dst[canonical(m)] = src[m]
__global__ void k_sc_permute(float* dst, const float* src, ScLayout L, bool to_internal) {
  for (uint32_t m = blockIdx.x * blockDim.x + threadIdx.x; m < L.n; m += gridDim.x * blockDim.x) {
    const uint32_t id = sc_canonical(L, m);
    if (to_internal) dst[m] = src[id]; else dst[id] = src[m];
  }
}

// ---- measurement --------------------------------------------------------------------------------
// block partial of (sum Sx, sum Sy, sum Sz, sum e_i) in double; partials[block*4 + q]
__device__ __forceinline__ void block_reduce4(double a0, double a1, double a2, double a3, double* partials) {
  __shared__ double sh[4][32];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    a0 += __shfl_xor_sync(0xffffffffu, a0, o);
    a1 += __shfl_xor_sync(0xffffffffu, a1, o);
    a2 += __shfl_xor_sync(0xffffffffu, a2, o);
    a3 += __shfl_xor_sync(0xffffffffu, a3, o);
  }
  const int w = threadIdx.x >> 5, l = threadIdx.x & 31, nw = (blockDim.x + 31) >> 5;
  if (l == 0) { sh[0][w] = a0; sh[1][w] = a1; sh[2][w] = a2; sh[3][w] = a3; }
  __syncthreads();
  if (w == 0) {
    a0 = l < nw ? sh[0][l] : 0.0; a1 = l < nw ? sh[1][l] : 0.0;
    a2 = l < nw ? sh[2][l] : 0.0; a3 = l < nw ? sh[3][l] : 0.0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      a0 += __shfl_xor_sync(0xffffffffu, a0, o);
      a1 += __shfl_xor_sync(0xffffffffu, a1, o);
      a2 += __shfl_xor_sync(0xffffffffu, a2, o);
      a3 += __shfl_xor_sync(0xffffffffu, a3, o);
    }
    if (l == 0) {
      partials[blockIdx.x * 4 + 0] = a0; partials[blockIdx.x * 4 + 1] = a1;
      partials[blockIdx.x * 4 + 2] = a2; partials[blockIdx.x * 4 + 3] = a3;
    }
  }
}

// fixed-order final sum of the block partials: one block of 256 threads
__global__ void k_reduce_final(const double* partials, int n_blocks, double* out) {
  double a[4] = {0, 0, 0, 0};
  for (int b = threadIdx.x; b < n_blocks; b += blockDim.x)
    for (int q = 0; q < 4; ++q) a[q] += partials[b * 4 + q];
  __shared__ double sh[4][256];
  for (int q = 0; q < 4; ++q) sh[q][threadIdx.x] = a[q];
  __syncthreads();
  for (int s = 128; s > 0; s >>= 1) {
    if ((int)threadIdx.x < s)
      for (int q = 0; q < 4; ++q) sh[q][threadIdx.x] += sh[q][threadIdx.x + s];
    __syncthreads();
  }
  if (threadIdx.x < 4) out[threadIdx.x] = sh[threadIdx.x][0];
}

template <int V>
__global__ void __launch_bounds__(256)
k_measure_sc(const float* __restrict__ sx, const float* __restrict__ sy, const float* __restrict__ sz,
             ScLayout L, SweepParams P, double* partials) {
  const uint32_t HV = (uint32_t)L.H / V;
  const uint32_t per_colour = (uint32_t)L.Lz * (uint32_t)L.Ly * HV;
  double mx = 0, my = 0, mz = 0, en = 0;
  for (uint32_t q = blockIdx.x * blockDim.x + threadIdx.x; q < 2u * per_colour; q += gridDim.x * blockDim.x) {
    const uint32_t c = q >= per_colour ? 1u : 0u;
    const uint32_t r = q - c * per_colour;
    const uint32_t row = r / HV, j = r - row * HV;
    const int32_t z = (int32_t)(row / (uint32_t)L.Ly), y = (int32_t)(row - (uint32_t)z * (uint32_t)L.Ly);
    const int32_t ym = (y == 0) ? L.Ly - 1 : y - 1, yp = (y == L.Ly - 1) ? 0 : y + 1;
    const int32_t zm = (z == 0) ? L.Lz - 1 : z - 1, zp = (z == L.Lz - 1) ? 0 : z + 1;
    const int32_t p = (int32_t)((c + (uint32_t)y + (uint32_t)z) & 1u), i0 = (int32_t)(j * V);
    const uint32_t row_c = row * (uint32_t)L.H;
    const uint32_t row_ym = (uint32_t)(z * L.Ly + ym) * L.H, row_yp = (uint32_t)(z * L.Ly + yp) * L.H;
    const uint32_t row_zm = (uint32_t)(zm * L.Ly + y) * L.H, row_zp = (uint32_t)(zp * L.Ly + y) * L.H;
    const uint32_t own = c * L.half, oth = (1u - c) * L.half;
    const Vec<V> hx = sc_field<V>(sx + oth, L, row_c, row_ym, row_yp, row_zm, row_zp, i0, p);
    const Vec<V> hy = sc_field<V>(sy + oth, L, row_c, row_ym, row_yp, row_zm, row_zp, i0, p);
    const Vec<V> hz = sc_field<V>(sz + oth, L, row_c, row_ym, row_yp, row_zm, row_zp, i0, p);
    const Vec<V> ox = load_ro<V>(sx + own + row_c + i0), oy = load_ro<V>(sy + own + row_c + i0),
                 oz = load_ro<V>(sz + own + row_c + i0);
#pragma unroll
    for (int k = 0; k < V; ++k) {
      mx += (double)ox.v[k]; my += (double)oy.v[k]; mz += (double)oz.v[k];
      en += (double)site_energy(ox.v[k], oy.v[k], oz.v[k], hx.v[k], hy.v[k], hz.v[k], P.J, P.K, P.ex, P.ey, P.ez);
    }
  }
  block_reduce4(mx, my, mz, en, partials);
}

__global__ void __launch_bounds__(256)
k_measure_csr(const float* __restrict__ sx, const float* __restrict__ sy, const float* __restrict__ sz,
              CsrDev g, SweepParams P, double* partials) {
  double mx = 0, my = 0, mz = 0, en = 0;
  for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < g.n; i += gridDim.x * blockDim.x) {
    const int32_t k0 = g.row_ptr[i], k1 = g.row_ptr[i + 1];
    float hx = 0.0f, hy = 0.0f, hz = 0.0f;
    for (int32_t k = k0; k < k1; ++k) {
      const int32_t j = __ldg(g.col + k);
      hx = __fadd_rn(hx, __ldg(sx + j));
      hy = __fadd_rn(hy, __ldg(sy + j));
      hz = __fadd_rn(hz, __ldg(sz + j));
    }
    float K = P.K, ex = P.ex, ey = P.ey, ez = P.ez;
    if (g.K_site) {
      K = __ldg(g.K_site + i);
      ex = __ldg(g.e_site + 3 * (size_t)i);
      ey = __ldg(g.e_site + 3 * (size_t)i + 1);
      ez = __ldg(g.e_site + 3 * (size_t)i + 2);
    }
    const float ox = __ldg(sx + i), oy = __ldg(sy + i), oz = __ldg(sz + i);
    mx += (double)ox; my += (double)oy; mz += (double)oz;
    en += (double)site_energy(ox, oy, oz, hx, hy, hz, P.J, K, ex, ey, ez);
  }
  block_reduce4(mx, my, mz, en, partials);
}

inline int grid_for(uint32_t n, int block, int cap) {
  const long long g = ((long long)n + block - 1) / block;
  return (int)(g < 1 ? 1 : (g > cap ? cap : g));
}

}  // namespace

// ---- launchers -----------------------------------------------------------------------------------
cudaError_t launch_init_random_sc(cudaStream_t st, float* s, ScLayout L, uint32_t seed_lo, uint32_t seed_hi) {
  k_init_random_sc<<<grid_for(L.n, 256, 148 * 16), 256, 0, st>>>(s, s + L.n, s + 2 * (size_t)L.n, L, seed_lo, seed_hi);
  return cudaGetLastError();
}

cudaError_t launch_init_random_flat(cudaStream_t st, float* s, uint32_t n, uint32_t seed_lo, uint32_t seed_hi) {
  k_init_random_flat<<<grid_for(n, 256, 148 * 16), 256, 0, st>>>(s, s + n, s + 2 * (size_t)n, n, seed_lo, seed_hi);
  return cudaGetLastError();
}

cudaError_t launch_fill(cudaStream_t st, float* s, uint32_t n, float x, float y, float z) {
  k_fill<<<grid_for(n, 256, 148 * 16), 256, 0, st>>>(s, s + n, s + 2 * (size_t)n, n, x, y, z);
  return cudaGetLastError();
}

cudaError_t launch_sc_permute(cudaStream_t st, float* dst, const float* src, ScLayout L, bool to_internal) {
  k_sc_permute<<<grid_for(L.n, 256, 148 * 16), 256, 0, st>>>(dst, src, L, to_internal);
  return cudaGetLastError();
}

template <int V, bool DIAG>
static cudaError_t sweep_sc_impl(cudaStream_t st, float* s, ScLayout L, ScTile t, SweepParams p, int colour, Diag d) {
  const size_t n = L.n;
  float* a = s + (size_t)colour * L.half;
  const float* b = s + (size_t)(1 - colour) * L.half;
  const int HV = L.H / V;
  dim3 grid((HV + t.JX - 1) / t.JX, (L.Ly + t.TY - 1) / t.TY, (L.Lz + t.ZT - 1) / t.ZT);
  k_sweep_sc<V, DIAG><<<grid, t.JX * t.TY, 0, st>>>(a, a + n, a + 2 * n, b, b + n, b + 2 * n, L, t, p, colour, d);
  return cudaGetLastError();
}

cudaError_t launch_sweep_sc(cudaStream_t st, float* s, ScLayout L, ScTile t, SweepParams p, int colour, Diag d) {
  const bool diag = d.accept || d.n_accept;
  switch (t.V) {
    case 4: return diag ? sweep_sc_impl<4, true>(st, s, L, t, p, colour, d) : sweep_sc_impl<4, false>(st, s, L, t, p, colour, d);
    case 2: return diag ? sweep_sc_impl<2, true>(st, s, L, t, p, colour, d) : sweep_sc_impl<2, false>(st, s, L, t, p, colour, d);
    default: return diag ? sweep_sc_impl<1, true>(st, s, L, t, p, colour, d) : sweep_sc_impl<1, false>(st, s, L, t, p, colour, d);
  }
}

cudaError_t launch_sweep_csr(cudaStream_t st, float* s, CsrDev g, uint32_t list_begin, uint32_t list_count,
                             SweepParams p, int block, Diag d) {
  if (list_count == 0) return cudaSuccess;
  const size_t n = g.n;
  const int grid = (int)((list_count + block - 1) / block);
  if (d.accept || d.n_accept)
    k_sweep_csr<true><<<grid, block, 0, st>>>(s, s + n, s + 2 * n, g, list_begin, list_count, p, d);
  else
    k_sweep_csr<false><<<grid, block, 0, st>>>(s, s + n, s + 2 * n, g, list_begin, list_count, p, d);
  return cudaGetLastError();
}

cudaError_t launch_measure_sc(cudaStream_t st, const float* s, ScLayout L, int V, SweepParams p, double* partials, double* out) {
  const size_t n = L.n;
  const int grid = grid_for(L.n / V, 256, kMeasureBlocks);
  switch (V) {
    case 4: k_measure_sc<4><<<grid, 256, 0, st>>>(s, s + n, s + 2 * n, L, p, partials); break;
    case 2: k_measure_sc<2><<<grid, 256, 0, st>>>(s, s + n, s + 2 * n, L, p, partials); break;
    default: k_measure_sc<1><<<grid, 256, 0, st>>>(s, s + n, s + 2 * n, L, p, partials); break;
  }
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  k_reduce_final<<<1, 256, 0, st>>>(partials, grid, out);
  return cudaGetLastError();
}

cudaError_t launch_measure_csr(cudaStream_t st, const float* s, CsrDev g, SweepParams p, double* partials, double* out) {
  const size_t n = g.n;
  const int grid = grid_for(g.n, 256, kMeasureBlocks);
  k_measure_csr<<<grid, 256, 0, st>>>(s, s + n, s + 2 * n, g, p, partials);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  k_reduce_final<<<1, 256, 0, st>>>(partials, grid, out);
  return cudaGetLastError();
}

}  // namespace hb
