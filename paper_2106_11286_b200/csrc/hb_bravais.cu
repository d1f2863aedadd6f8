// hb_bravais.cu -- colour kernels for periodic Bravais lattices with a basis (bcc, fcc), implicit
// neighbour indexing: no neighbour table is read, the geometry is a compile-time descriptor.
//
// Storage is the canonical order: sublattice b is a plain Lx x Ly x Lz array at
// offset b*Nc of each component plane, and colour = b.  A thread owns V consecutive cells of one
// x-row of its sublattice and marches ZT planes in z, exactly like the sc kernel; a neighbour of
// the V cells [i0, i0+V) of row (y,z) is the same V-vector of another sublattice's row
// (y+dy, z+dz), shifted by dx in {-1,0,+1}: one aligned vector load plus, for dx != 0, one halo
// element.  Neighbours that share a row share the loads (the compiler merges them; ptxas output
// is checked in profiles/).  Neighbour order is the arithmetic contract of include/hb.h.
//
// HBM traffic per attempted update: bcc 36 B (own 12 + other sublattice once 12 + write 12),
// fcc 60 B (own 12 + three other sublattices 36 + write 12); DESIGN.md section 7.
#include "hb_device.cuh"
#include "hb_internal.h"
#include "hb_bravais_geo.cuh"

namespace hb {

namespace {

// what a thread knows about its V cells in row (y,z): element offsets inside one sublattice array
// resident 256-thread blocks per SM the plain pass is compiled for: fcc runs 5 % faster with four (64 registers, 16-24 bytes of
// spills: its 36 neighbour loads per thread and plane want warps more than registers: c3 80.0 -> 84.3 Gupd/s), bcc 3 % slower
#ifndef HB_FCC_MINBLOCKS
#define HB_FCC_MINBLOCKS 4
#endif
template <int KIND> __host__ __device__ constexpr int br_min_blocks() { return KIND == BR_FCC ? HB_FCC_MINBLOCKS : 3; }
struct Where {
  uint32_t yo[3];   // (y-1, y, y+1 periodic) * Lx
  uint32_t zo[3];   // (z-1, z, z+1 periodic) * Ly * Lx
  uint32_t i0, il, ir;   // first cell, the cell left of it and the cell right of the last one (periodic)
};

template <int V>
__device__ __forceinline__ Vec<V> shifted(const float* __restrict__ row, const Where& w, int dx) {
  const Vec<V> c = load_ro<V>(row + w.i0);
  if (dx == 0) return c;
  Vec<V> t;
  if (dx < 0) {
    t.v[0] = __ldg(row + w.il);
#pragma unroll
    for (int k = 1; k < V; ++k) t.v[k] = c.v[k - 1];
  } else {
#pragma unroll
    for (int k = 0; k + 1 < V; ++k) t.v[k] = c.v[k + 1];
    t.v[V - 1] = __ldg(row + w.ir);
  }
  return t;
}

template <int V>
__device__ __forceinline__ Vec<V> vadd(const Vec<V>& a, const Vec<V>& b) {
  Vec<V> r;
  if (V >= 2) {
#pragma unroll
    for (int k = 0; k + 1 < V; k += 2) {
      const f2 s = add2(make_float2(a.v[k], a.v[k + 1]), make_float2(b.v[k], b.v[k + 1]));
      r.v[k] = s.x; r.v[k + 1] = s.y;
    }
  } else {
    r.v[0] = __fadd_rn(a.v[0], b.v[0]);
  }
  return r;
}

// h = sum over the Z neighbours in contract order, starting from the first one (0 + a = a exactly)
template <int KIND, int B, int V, int K = 0>
__device__ __forceinline__ void field(const float* __restrict__ s, uint32_t nc, uint32_t n, const Where& w,
                                      Vec<V>& hx, Vec<V>& hy, Vec<V>& hz) {
  if constexpr (K < Geo<KIND>::Z) {
    constexpr Nbr g = Geo<KIND>::nbr(B, K);
    const float* row = s + (size_t)g.nb * nc + (w.zo[g.dz + 1] + w.yo[g.dy + 1]);
    const Vec<V> tx = shifted<V>(row, w, g.dx);
    const Vec<V> ty = shifted<V>(row + n, w, g.dx);
    const Vec<V> tz = shifted<V>(row + 2 * (size_t)n, w, g.dx);
    if constexpr (K == 0) { hx = tx; hy = ty; hz = tz; }
    else { hx = vadd<V>(hx, tx); hy = vadd<V>(hy, ty); hz = vadd<V>(hz, tz); }
    field<KIND, B, V, K + 1>(s, nc, n, w, hx, hy, hz);
  }
}

// the part of the field that comes from LOWER sublattices (colours already final in this sweep): with it every
// bond is charged exactly once, at its higher-colour end, for the fused measurement
template <int KIND, int B, int V, int K = 0>
__device__ __forceinline__ void field_low(const float* __restrict__ s, uint32_t nc, uint32_t n, const Where& w,
                                          Vec<V>& hx, Vec<V>& hy, Vec<V>& hz) {
  if constexpr (K == 0) {
#pragma unroll
    for (int k = 0; k < V; ++k) { hx.v[k] = 0.0f; hy.v[k] = 0.0f; hz.v[k] = 0.0f; }
  }
  if constexpr (K < Geo<KIND>::Z) {
    constexpr Nbr g = Geo<KIND>::nbr(B, K);
    if constexpr (g.nb < B) {
      const float* row = s + (size_t)g.nb * nc + (w.zo[g.dz + 1] + w.yo[g.dy + 1]);
      hx = vadd<V>(hx, shifted<V>(row, w, g.dx));
      hy = vadd<V>(hy, shifted<V>(row + n, w, g.dx));
      hz = vadd<V>(hz, shifted<V>(row + 2 * (size_t)n, w, g.dx));
    }
    field_low<KIND, B, V, K + 1>(s, nc, n, w, hx, hy, hz);
  }
}

__device__ __forceinline__ void where_y(Where& w, const BrLayout& L, int32_t y, int32_t i0, int V) {
  w.yo[0] = (uint32_t)((y == 0) ? L.Ly - 1 : y - 1) * (uint32_t)L.Lx;
  w.yo[1] = (uint32_t)y * (uint32_t)L.Lx;
  w.yo[2] = (uint32_t)((y == L.Ly - 1) ? 0 : y + 1) * (uint32_t)L.Lx;
  w.i0 = (uint32_t)i0;
  w.il = (uint32_t)((i0 == 0) ? L.Lx - 1 : i0 - 1);
  w.ir = (uint32_t)((i0 + V >= L.Lx) ? i0 + V - L.Lx : i0 + V);
}
__device__ __forceinline__ void where_z(Where& w, const BrLayout& L, int32_t z) {
  const uint32_t plane = (uint32_t)L.Ly * (uint32_t)L.Lx;
  w.zo[0] = (uint32_t)((z == 0) ? L.Lz - 1 : z - 1) * plane;
  w.zo[1] = (uint32_t)z * plane;
  w.zo[2] = (uint32_t)((z == L.Lz - 1) ? 0 : z + 1) * plane;
}

template <int KIND, int B, int V, int ANISO, bool DIAG, bool MEAS = false>
__global__ void __launch_bounds__(256, (MEAS && n_low<KIND, B>() != 0 && n_low<KIND, B>() != Geo<KIND>::Z) ? 1 : (MEAS ? 2 : br_min_blocks<KIND>()))
k_sweep_bravais(float* __restrict__ own, const float* __restrict__ all, BrLayout L, ScTile t, SweepParams P, Diag d, Meas m) {
  resolve_sweep(P);
  const int32_t tj = threadIdx.x % t.JX, ty = threadIdx.x / t.JX;
  const int32_t i0 = (blockIdx.x * t.JX + tj) * V;
  const int32_t y = blockIdx.y * t.TY + ty;
  const bool outside = i0 >= L.Lx || y >= L.Ly;
  if (!MEAS && outside) return;
  Where w;
  where_y(w, L, outside ? 0 : y, outside ? 0 : i0, V);
  const int32_t z0 = blockIdx.z * t.ZT, z1 = (MEAS && outside) ? z0 : min(z0 + t.ZT, L.Lz);
  const size_t n = L.n;
  unsigned n_acc = 0;
  double acc_mx = 0.0, acc_my = 0.0, acc_mz = 0.0, acc_en = 0.0;
  for (int32_t z = z0; z < z1; ++z) {
    if (L.ghost && (z == 0 || z == L.Lz - 1)) continue;      // ghost planes of a slab: the z-neighbour owns them
    where_z(w, L, z);
    const uint32_t o = w.zo[1] + w.yo[1] + w.i0;             // offset inside the own sublattice
    Vec<V> sx = load_rw<V>(own + o), sy = load_rw<V>(own + n + o), sz = load_rw<V>(own + 2 * n + o);
    Vec<V> hx, hy, hz;
    field<KIND, B, V>(all, L.nc, L.n, w, hx, hy, hz);
    const uint32_t site0 = (uint32_t)B * L.nc_id + o + L.cell_base;   // canonical id = b*Nc + cell (of the whole lattice)
    bool any = false;
    if constexpr (V >= 2) {
#pragma unroll
      for (int k = 0; k + 1 < V; k += 2) {
        const Rand4 ra = philox4x32_10(site0 + k, 0u, P.sweep_lo, P.sweep_hi, P.seed_lo, P.seed_hi);
        const Rand4 rb = philox4x32_10(site0 + k + 1, 0u, P.sweep_lo, P.sweep_hi, P.seed_lo, P.seed_hi);
        f2 px = make_float2(sx.v[k], sx.v[k + 1]), py = make_float2(sy.v[k], sy.v[k + 1]), pz = make_float2(sz.v[k], sz.v[k + 1]);
        bool acc_a, acc_b;
        attempt2<ANISO>(ra, rb, P.J, P.K, P.beta, P.ex, P.ey, P.ez, make_float2(hx.v[k], hx.v[k + 1]),
                        make_float2(hy.v[k], hy.v[k + 1]), make_float2(hz.v[k], hz.v[k + 1]), px, py, pz, acc_a, acc_b);
        sx.v[k] = px.x; sx.v[k + 1] = px.y; sy.v[k] = py.x; sy.v[k + 1] = py.y; sz.v[k] = pz.x; sz.v[k + 1] = pz.y;
        any |= acc_a | acc_b;
        if (DIAG || MEAS) n_acc += (unsigned)acc_a + (unsigned)acc_b;
        if (DIAG) {
          if (d.accept) { d.accept[site0 + k] = acc_a; d.accept[site0 + k + 1] = acc_b; }
        }
      }
    } else {
      const Rand4 r = philox4x32_10(site0, 0u, P.sweep_lo, P.sweep_hi, P.seed_lo, P.seed_hi);
      float nx, ny, nz;
      sphere(r.r0, r.r1, nx, ny, nz);
      const float dH = delta_h_t<ANISO>(sx.v[0], sy.v[0], sz.v[0], nx, ny, nz, hx.v[0], hy.v[0], hz.v[0], P.J, P.K, P.ex, P.ey, P.ez);
      const bool acc = metropolis_accept(dH, P.beta, r.r2);
      if (acc) { sx.v[0] = nx; sy.v[0] = ny; sz.v[0] = nz; }
      any = acc;
      if (DIAG || MEAS) n_acc += acc;
      if (DIAG) {
        if (d.accept) d.accept[site0] = acc;
      }
    }
    if (any) {
      store<V>(own + o, sx);
      store<V>(own + n + o, sy);
      store<V>(own + 2 * n + o, sz);
    }
    if (MEAS) {
      Vec<V> lx, ly, lz;
      if constexpr (n_low<KIND, B>() == Geo<KIND>::Z) { lx = hx; ly = hy; lz = hz; }   // highest colour: the whole field
      else field_low<KIND, B, V>(all, L.nc, L.n, w, lx, ly, lz);
      float gx = 0.0f, gy = 0.0f, gz = 0.0f, ge = 0.0f;
#pragma unroll
      for (int k = 0; k < V; ++k) {
        gx = __fadd_rn(gx, sx.v[k]); gy = __fadd_rn(gy, sy.v[k]); gz = __fadd_rn(gz, sz.v[k]);
        const float sl = __fmaf_rn(sz.v[k], lz.v[k], __fmaf_rn(sy.v[k], ly.v[k], __fmul_rn(sx.v[k], lx.v[k])));
        const float a = __fmaf_rn(sz.v[k], P.ez, __fmaf_rn(sy.v[k], P.ey, __fmul_rn(sx.v[k], P.ex)));
        ge = __fadd_rn(ge, __fmaf_rn(-P.J, sl, __fmul_rn(-P.K, __fmul_rn(a, a))));
      }
      acc_mx += (double)gx; acc_my += (double)gy; acc_mz += (double)gz; acc_en += (double)ge;
    }
  }
  if (DIAG && d.n_accept && n_acc) atomicAdd(d.n_accept, (unsigned long long)n_acc);
  if (MEAS) {
    const uint32_t blk = (blockIdx.z * gridDim.y + blockIdx.y) * gridDim.x + blockIdx.x;
    block_reduce4(acc_mx, acc_my, acc_mz, acc_en, m.partials + (size_t)blk * 4);
    if (!DIAG) count_accepts(m.n_accept, n_acc);
  }
}

// ---- measurement: M and E over all sublattices, fp64 accumulation ---------------------------------
template <int KIND, int B, int V>
__device__ __forceinline__ void measure_sub(const float* __restrict__ s, const BrLayout& L, const SweepParams& P,
                                            double& mx, double& my, double& mz, double& en) {
  if constexpr (B < Geo<KIND>::NB) {
    const uint32_t HV = (uint32_t)L.Lx / V, chunks = (uint32_t)L.Lz * (uint32_t)L.Ly * HV;
    const size_t n = L.n;
    for (uint32_t q = blockIdx.x * blockDim.x + threadIdx.x; q < chunks; q += gridDim.x * blockDim.x) {
      const uint32_t row = q / HV, j = q - row * HV;
      const int32_t z = (int32_t)(row / (uint32_t)L.Ly), y = (int32_t)(row - (uint32_t)z * (uint32_t)L.Ly);
      if (L.ghost && (z == 0 || z == L.Lz - 1)) continue;    // a slab sums its own planes only
      Where w;
      where_y(w, L, y, (int32_t)(j * V), V);
      where_z(w, L, z);
      Vec<V> hx, hy, hz;
      field<KIND, B, V>(s, L.nc, L.n, w, hx, hy, hz);
      const float* own = s + (size_t)B * L.nc + (w.zo[1] + w.yo[1] + w.i0);
      const Vec<V> ox = load_ro<V>(own), oy = load_ro<V>(own + n), oz = load_ro<V>(own + 2 * n);
#pragma unroll
      for (int k = 0; k < V; ++k) {
        mx += (double)ox.v[k]; my += (double)oy.v[k]; mz += (double)oz.v[k];
        en += (double)site_energy(ox.v[k], oy.v[k], oz.v[k], hx.v[k], hy.v[k], hz.v[k], P.J, P.K, P.ex, P.ey, P.ez);
      }
    }
    measure_sub<KIND, B + 1, V>(s, L, P, mx, my, mz, en);
  }
}

template <int KIND, int V>
__global__ void __launch_bounds__(256)
k_measure_bravais(const float* __restrict__ s, BrLayout L, SweepParams P, double* partials) {
  double mx = 0, my = 0, mz = 0, en = 0;
  measure_sub<KIND, 0, V>(s, L, P, mx, my, mz, en);
  block_reduce4(mx, my, mz, en, partials + (size_t)blockIdx.x * 4);
}

__global__ void k_init_random_bravais(float* sx, float* sy, float* sz, BrLayout L, uint32_t seed_lo, uint32_t seed_hi) {
  for (unsigned long long m64 = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; m64 < L.n; m64 += (unsigned long long)gridDim.x * blockDim.x) {
    const uint32_t m = (uint32_t)m64, b = m / L.nc, q = m - b * L.nc;
    const Rand4 r = philox4x32_10(b * L.nc_id + q + L.cell_base, 1u, 0u, 0u, seed_lo, seed_hi);
    float x, y, z;
    sphere(r.r0, r.r1, x, y, z);
    sx[m] = x; sy[m] = y; sz[m] = z;
  }
}

inline int aniso_of(const SweepParams& p) {
  return (p.K == 0.0f) ? ANISO_NONE : ((p.ex == 0.0f && p.ey == 0.0f && p.ez == 1.0f) ? ANISO_Z : ANISO_GENERAL);
}

template <int KIND, int B, int V, int ANISO, bool DIAG, bool MEAS = false>
cudaError_t go(cudaStream_t st, float* s, const BrLayout& L, const ScTile& t, const SweepParams& p, const Diag& d,
               const Meas& m = Meas{nullptr, 0, nullptr}) {
  const int HV = L.Lx / V;
  dim3 grid((HV + t.JX - 1) / t.JX, (L.Ly + t.TY - 1) / t.TY, (L.Lz + t.ZT - 1) / t.ZT);
  return launch_colour_kernel(k_sweep_bravais<KIND, B, V, ANISO, DIAG, MEAS>, grid, dim3(t.JX * t.TY), 0, st, p.pdl != 0,
                              s + (size_t)B * L.nc, s, L, t, p, d, m);
}

// The tuned shape (V = 4, no diagnostics) carries the three anisotropy specialisations; the
// narrow vectors and the recording variant use the general formula, which gives the same bits.
template <int KIND, int B>
cudaError_t pick(cudaStream_t st, float* s, const BrLayout& L, const ScTile& t, const SweepParams& p, const Diag& d, const Meas& m) {
  const bool diag = d.accept || d.n_accept;
  if (m.mode != 0) {   // fused measurement: tuned vector width only, general anisotropy formula (same bits)
    if (t.V != 4 || diag) return cudaErrorInvalidValue;
    return go<KIND, B, 4, ANISO_GENERAL, false, true>(st, s, L, t, p, d, m);
  }
  if (t.V == 4) {
    if (diag) return go<KIND, B, 4, ANISO_GENERAL, true>(st, s, L, t, p, d);
    switch (aniso_of(p)) {
      case ANISO_NONE: return go<KIND, B, 4, ANISO_NONE, false>(st, s, L, t, p, d);
      case ANISO_Z: return go<KIND, B, 4, ANISO_Z, false>(st, s, L, t, p, d);
      default: return go<KIND, B, 4, ANISO_GENERAL, false>(st, s, L, t, p, d);
    }
  }
  if (t.V == 2)
    return diag ? go<KIND, B, 2, ANISO_GENERAL, true>(st, s, L, t, p, d) : go<KIND, B, 2, ANISO_GENERAL, false>(st, s, L, t, p, d);
  return diag ? go<KIND, B, 1, ANISO_GENERAL, true>(st, s, L, t, p, d) : go<KIND, B, 1, ANISO_GENERAL, false>(st, s, L, t, p, d);
}

template <int KIND>
cudaError_t measure(cudaStream_t st, const float* s, const BrLayout& L, int V, const SweepParams& p, double* partials, int grid) {
  switch (V) {
    case 4: k_measure_bravais<KIND, 4><<<grid, 256, 0, st>>>(s, L, p, partials); break;
    case 2: k_measure_bravais<KIND, 2><<<grid, 256, 0, st>>>(s, L, p, partials); break;
    default: k_measure_bravais<KIND, 1><<<grid, 256, 0, st>>>(s, L, p, partials); break;
  }
  return cudaGetLastError();
}

}  // namespace

// blocks of one colour launch if it can carry the fused measurement (4 doubles of partials per block), else 0
int bravais_fused_blocks(const BrLayout& L, const ScTile& t) {
  if (t.V != 4) return 0;
  const int HV = L.Lx / 4;
  const long long blocks = (long long)((HV + t.JX - 1) / t.JX) * ((L.Ly + t.TY - 1) / t.TY) * ((L.Lz + t.ZT - 1) / t.ZT);
  return blocks <= kFusedBlocksMax / 2 ? (int)blocks : 0;   // four colours share the partials buffer
}

cudaError_t launch_sweep_bravais(cudaStream_t st, float* s, BrLayout L, ScTile t, SweepParams p, int colour, Diag d, Meas m) {
  if (L.kind == BR_BCC) {
    switch (colour) {
      case 0: return pick<BR_BCC, 0>(st, s, L, t, p, d, m);
      case 1: return pick<BR_BCC, 1>(st, s, L, t, p, d, m);
    }
  } else if (L.kind == BR_FCC) {
    switch (colour) {
      case 0: return pick<BR_FCC, 0>(st, s, L, t, p, d, m);
      case 1: return pick<BR_FCC, 1>(st, s, L, t, p, d, m);
      case 2: return pick<BR_FCC, 2>(st, s, L, t, p, d, m);
      case 3: return pick<BR_FCC, 3>(st, s, L, t, p, d, m);
    }
  }
  return cudaErrorInvalidValue;
}

cudaError_t launch_init_random_bravais(cudaStream_t st, float* s, BrLayout L, uint32_t seed_lo, uint32_t seed_hi) {
  const long long g = ((long long)L.n + 255) / 256;
  k_init_random_bravais<<<(unsigned)(g < 1 ? 1 : (g > 148 * 16 ? 148 * 16 : g)), 256, 0, st>>>(s, s + L.n, s + 2 * (size_t)L.n, L, seed_lo, seed_hi);
  return cudaGetLastError();
}

cudaError_t launch_measure_bravais(cudaStream_t st, const float* s, BrLayout L, int V, SweepParams p, double* partials, double* out) {
  const long long chunks = (long long)L.nc / V;
  const long long want = (chunks + 255) / 256;
  const int grid = (int)(want < 1 ? 1 : (want > kMeasureBlocks ? kMeasureBlocks : want));
  cudaError_t e = L.kind == BR_BCC ? measure<BR_BCC>(st, s, L, V, p, partials, grid) : measure<BR_FCC>(st, s, L, V, p, partials, grid);
  if (e != cudaSuccess) return e;
  return launch_reduce_final(st, partials, grid, out);
}

}  // namespace hb
