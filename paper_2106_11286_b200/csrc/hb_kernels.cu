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
#include <cooperative_groups.h>

#include "hb_device.cuh"
#include "hb_internal.h"

namespace hb {

namespace {

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
template <int ANISO = ANISO_GENERAL>
__device__ __forceinline__ bool attempt(uint32_t site, const SweepParams& P, float K, float ex, float ey, float ez,
                                        float hx, float hy, float hz, float& sx, float& sy, float& sz) {
  const Rand4 r = philox4x32_10(site, 0u, P.sweep_lo, P.sweep_hi, P.seed_lo, P.seed_hi);
  float nx, ny, nz;
  sphere(r.r0, r.r1, nx, ny, nz);
  const float dH = delta_h_t<ANISO>(sx, sy, sz, nx, ny, nz, hx, hy, hz, P.J, K, ex, ey, ez);
  const bool acc = metropolis_accept(dH, P.beta, r.r2);
  sx = acc ? nx : sx;
  sy = acc ? ny : sy;
  sz = acc ? nz : sz;
  return acc;
}

#ifndef HB_SC_MINBLOCKS
#define HB_SC_MINBLOCKS 4
#endif
// Software prefetch of the lines the NEXT z-plane of the march touches for the first time:
// PF 0 none, 1 prefetch.global.L2, 2 prefetch.global.L1, 3 a real load into a register nobody reads.
template <int PF>
__device__ __forceinline__ void prefetch_line(const float* p) {
  if (PF == 1) asm volatile("prefetch.global.L2 [%0];" ::"l"(p));
  if (PF == 2) asm volatile("prefetch.global.L1 [%0];" ::"l"(p));
  if (PF == 3) { float t; asm volatile("ld.global.ca.f32 %0, [%1];" : "=f"(t) : "l"(p)); }
}

// Neighbour field from 32-bit element offsets into one component plane of the other colour.
template <int V, bool CO = false>
__device__ __forceinline__ Vec<V> sc_field_off(const float* b, uint32_t oc, uint32_t oh, uint32_t oym,
                                               uint32_t oyp, uint32_t ozm, uint32_t ozp, int32_t p) {
  const Vec<V> c = CO ? load_co<V>(b + oc) : load_ro<V>(b + oc);
  const float halo = CO ? __ldca(b + oh) : __ldg(b + oh);
  const Vec<V> ym = CO ? load_co<V>(b + oym) : load_ro<V>(b + oym);
  const Vec<V> yp = CO ? load_co<V>(b + oyp) : load_ro<V>(b + oyp);
  const Vec<V> zm = CO ? load_co<V>(b + ozm) : load_ro<V>(b + ozm);
  const Vec<V> zp = CO ? load_co<V>(b + ozp) : load_ro<V>(b + ozp);
  Vec<V> h;
  if (V >= 2) {           // packed fp32x2 adds: same rounding per element, half the instructions
#pragma unroll
    for (int k = 0; k + 1 < V; k += 2) {
      const float lo0 = (k == 0) ? halo : c.v[k > 0 ? k - 1 : 0], lo1 = c.v[k];
      const float hi0 = c.v[k + 1], hi1 = (k + 1 == V - 1) ? halo : c.v[k + 2 < V ? k + 2 : 0];
      f2 s2 = add2(make_float2(c.v[k], c.v[k + 1]), make_float2(p ? hi0 : lo0, p ? hi1 : lo1));
      s2 = add2(s2, make_float2(ym.v[k], ym.v[k + 1]));
      s2 = add2(s2, make_float2(yp.v[k], yp.v[k + 1]));
      s2 = add2(s2, make_float2(zm.v[k], zm.v[k + 1]));
      s2 = add2(s2, make_float2(zp.v[k], zp.v[k + 1]));
      h.v[k] = s2.x; h.v[k + 1] = s2.y;
    }
  } else {
    float s = __fadd_rn(c.v[0], halo);
    s = __fadd_rn(s, ym.v[0]);
    s = __fadd_rn(s, yp.v[0]);
    s = __fadd_rn(s, zm.v[0]);
    s = __fadd_rn(s, zp.v[0]);
    h.v[0] = s;
  }
  return h;
}

// MEAS: the pass also reduces what a measurement needs from the spins it has just decided (SURVEY 8(a)
// note on fusing a5 into a4): every colour adds its own final spins to M and its anisotropy energy;
// the LAST colour (m.mode == 2) sees only final neighbours, and since every bond of a 2-colour lattice
// has exactly one end in it, -J sum_{i in last colour} S_i.h_i is the whole exchange energy.
// The pass of one block (bid of nblk): the body of k_sweep_sc, and of the persistent multi-sweep kernel below,
// which walks virtual blocks and needs coherent loads (CO) because other blocks of the same launch wrote b.
// SLAB: first and last planes are ghost planes of a slab (not updated), boundary-plane stores are repeated into the
// z-neighbours' buffers (hb_slab_set_peer); a separate instantiation, so that whole lattices carry none of it
template <int V, int ANISO, bool DIAG, int PF, bool MEAS, bool CO, bool SLAB = false>
__device__ __forceinline__ void sc_pass(float* ax, float* ay, float* az, const float* bx, const float* by, const float* bz,
                                        const ScLayout& L, const ScTile& t, const SweepParams& P, int colour, const Diag& d,
                                        const Meas& m, const uint3 bid, const uint3 nblk) {
  int32_t j, y, zl = -1;
  if (t.LIN < 0) {
    // whole colour pass in ONE block (tiny lattices): thread = one (z, y, x-vector) slot
    const int32_t HV = L.H / V;
    const uint32_t s = threadIdx.x;
    j = (int32_t)(s % (uint32_t)HV);
    y = (int32_t)((s / (uint32_t)HV) % (uint32_t)L.Ly);
    zl = (int32_t)(s / (uint32_t)(HV * L.Ly));
  } else if (t.LIN) {
    // linear mapping: the block owns blockDim.x consecutive (y, j) slots, so every warp is full
    // even when a row does not hold a multiple of 32 vectors (L = 464: 116 vectors per row)
    const int32_t HV = L.H / V;
    const uint32_t s = bid.x * blockDim.x + threadIdx.x;
    y = (int32_t)(s / (uint32_t)HV);
    j = (int32_t)(s - (uint32_t)y * (uint32_t)HV);
  } else {
    const int32_t tj = threadIdx.x % t.JX, ty = threadIdx.x / t.JX;
    j = (int32_t)bid.x * t.JX + tj;
    y = (int32_t)bid.y * t.TY + ty;
  }
  const int32_t i0 = j * V;
  const bool outside = i0 >= L.H || y >= L.Ly || zl >= L.Lz;
  if (!MEAS && outside) return;
  const uint32_t H = (uint32_t)L.H, plane = (uint32_t)L.Ly * H;
  const uint32_t ym = (uint32_t)((y == 0) ? L.Ly - 1 : y - 1) * H + (uint32_t)i0;
  const uint32_t yp = (uint32_t)((y == L.Ly - 1) ? 0 : y + 1) * H + (uint32_t)i0;
  const uint32_t yc = (uint32_t)y * H + (uint32_t)i0;
  const int32_t z0 = zl >= 0 ? zl : (int32_t)bid.z * t.ZT;
  const int32_t z1 = (MEAS && outside) ? z0 : (zl >= 0 ? zl + 1 : min(z0 + t.ZT, L.Lz));   // MEAS: every thread reaches the block reduction
  unsigned n_acc = 0;
  double acc_mx = 0.0, acc_my = 0.0, acc_mz = 0.0, acc_en = 0.0;
  for (int32_t z = z0; z < z1; ++z) {
    if (SLAB && (z == 0 || z == L.Lz - 1)) continue;   // ghost planes of a slab: the z-neighbour owns them
    const uint32_t pz = (uint32_t)z * plane;
    const uint32_t pzm = (uint32_t)((z == 0) ? L.Lz - 1 : z - 1) * plane;
    const uint32_t pzp = (uint32_t)((z == L.Lz - 1) ? 0 : z + 1) * plane;
    const int32_t p = (colour + y + z) & 1;
    int32_t ih = p ? V : -1;                          // the one element outside [i0, i0+V), periodic in x
    ih = (i0 + ih < 0) ? ih + L.H : ((i0 + ih >= L.H) ? ih - L.H : ih);
    const uint32_t oc = pz + yc, oh = oc + (uint32_t)ih, oym = pz + ym, oyp = pz + yp, ozm = pzm + yc, ozp = pzp + yc;
    Vec<V> sx = load_rw<V>(ax + oc), sy = load_rw<V>(ay + oc), sz = load_rw<V>(az + oc);
    const Vec<V> hx = sc_field_off<V, CO>(bx, oc, oh, oym, oyp, ozm, ozp, p);
    const Vec<V> hy = sc_field_off<V, CO>(by, oc, oh, oym, oyp, ozm, ozp, p);
    const Vec<V> hz = sc_field_off<V, CO>(bz, oc, oh, oym, oyp, ozm, ozp, p);
    if (PF != 0 && z + 1 < z1) {
      const uint32_t zpp = (uint32_t)((z + 2 >= L.Lz) ? z + 2 - L.Lz : z + 2) * plane + yc;
      prefetch_line<PF>(ax + pzp + yc); prefetch_line<PF>(ay + pzp + yc); prefetch_line<PF>(az + pzp + yc);
      prefetch_line<PF>(bx + pzp + ym); prefetch_line<PF>(by + pzp + ym); prefetch_line<PF>(bz + pzp + ym);
      prefetch_line<PF>(bx + pzp + yp); prefetch_line<PF>(by + pzp + yp); prefetch_line<PF>(bz + pzp + yp);
      prefetch_line<PF>(bx + zpp); prefetch_line<PF>(by + zpp); prefetch_line<PF>(bz + zpp);
    }
    const uint32_t site0 = (uint32_t)(z * L.Ly + y) * (uint32_t)L.Lx + 2u * (uint32_t)i0 + (uint32_t)p + L.site_base;
    bool any = false;
    if (V >= 2) {
#pragma unroll
      for (int k = 0; k + 1 < V; k += 2) {
        const Rand4 ra = philox4x32_10(site0 + 2u * k, 0u, P.sweep_lo, P.sweep_hi, P.seed_lo, P.seed_hi);
        const Rand4 rb = philox4x32_10(site0 + 2u * k + 2u, 0u, P.sweep_lo, P.sweep_hi, P.seed_lo, P.seed_hi);
        f2 px = make_float2(sx.v[k], sx.v[k + 1]), py = make_float2(sy.v[k], sy.v[k + 1]), pz = make_float2(sz.v[k], sz.v[k + 1]);
        bool acc_a, acc_b;
        attempt2<ANISO>(ra, rb, P.J, P.K, P.beta, P.ex, P.ey, P.ez, make_float2(hx.v[k], hx.v[k + 1]),
                        make_float2(hy.v[k], hy.v[k + 1]), make_float2(hz.v[k], hz.v[k + 1]), px, py, pz, acc_a, acc_b);
        sx.v[k] = px.x; sx.v[k + 1] = px.y; sy.v[k] = py.x; sy.v[k + 1] = py.y; sz.v[k] = pz.x; sz.v[k + 1] = pz.y;
        any |= acc_a | acc_b;
        if (DIAG || MEAS) n_acc += (unsigned)acc_a + (unsigned)acc_b;
        if (DIAG) {
          if (d.accept) { d.accept[site0 + 2u * k] = acc_a; d.accept[site0 + 2u * k + 2u] = acc_b; }
        }
      }
    } else {
      const bool acc = attempt<ANISO>(site0, P, P.K, P.ex, P.ey, P.ez, hx.v[0], hy.v[0], hz.v[0], sx.v[0], sy.v[0], sz.v[0]);
      any |= acc;
      if (DIAG || MEAS) n_acc += acc;
      if (DIAG) {
        if (d.accept) d.accept[site0] = acc;
      }
    }
    if (any) {
      store<V>(ax + oc, sx);
      store<V>(ay + oc, sy);
      store<V>(az + oc, sz);
      if (SLAB) {   // slab with peer stores: the boundary planes go straight into the neighbours' ghost planes
        const bool lo = z == 1, hi = z == L.Lz - 2;   // (distinct planes: a slab has at least two of its own)
        float* pb = lo ? L.peer[0] : (hi ? L.peer[1] : nullptr);
        if (pb) {
          const uint32_t pn = lo ? L.peer_n[0] : L.peer_n[1], ph = lo ? L.peer_half[0] : L.peer_half[1];
          float* q = pb + (size_t)colour * ph + (lo ? L.peer_zoff[0] : L.peer_zoff[1]) + yc;
          store<V>(q, sx);
          store<V>(q + pn, sy);
          store<V>(q + 2 * (size_t)pn, sz);
        }
      }
    }
    if (MEAS) {
      // fp32 per-site terms, summed over the thread's V sites in fp32, accumulated in fp64
      float gx = 0.0f, gy = 0.0f, gz = 0.0f, ge = 0.0f;
      const float Jx = (m.mode == 2) ? -P.J : 0.0f;
#pragma unroll
      for (int k = 0; k < V; ++k) {
        gx = __fadd_rn(gx, sx.v[k]); gy = __fadd_rn(gy, sy.v[k]); gz = __fadd_rn(gz, sz.v[k]);
        const float sh = __fmaf_rn(sz.v[k], hz.v[k], __fmaf_rn(sy.v[k], hy.v[k], __fmul_rn(sx.v[k], hx.v[k])));
        const float a = __fmaf_rn(sz.v[k], P.ez, __fmaf_rn(sy.v[k], P.ey, __fmul_rn(sx.v[k], P.ex)));
        ge = __fadd_rn(ge, __fmaf_rn(Jx, sh, __fmul_rn(-P.K, __fmul_rn(a, a))));
      }
      acc_mx += (double)gx; acc_my += (double)gy; acc_mz += (double)gz; acc_en += (double)ge;
    }
  }
  if (DIAG && d.n_accept && n_acc) atomicAdd(d.n_accept, (unsigned long long)n_acc);
  if (MEAS) {
    const uint32_t blk = (bid.z * nblk.y + bid.y) * nblk.x + bid.x;
    block_reduce4(acc_mx, acc_my, acc_mz, acc_en, m.partials + (size_t)blk * 4);
    if (!DIAG) count_accepts(m.n_accept, n_acc);
  }
}

template <int V, int ANISO, bool DIAG, int PF, int BLK = 256, bool MEAS = false, bool SLAB = false>
__global__ void __launch_bounds__(BLK, (MEAS ? 3 : HB_SC_MINBLOCKS) * 256 / BLK)   // MEAS needs ~80 registers
k_sweep_sc(float* __restrict__ ax, float* __restrict__ ay, float* __restrict__ az,
           const float* __restrict__ bx, const float* __restrict__ by, const float* __restrict__ bz,
           ScLayout L, ScTile t, SweepParams P, int colour, Diag d, Meas m) {
  resolve_sweep(P);
  sc_pass<V, ANISO, DIAG, PF, MEAS, false, SLAB>(ax, ay, az, bx, by, bz, L, t, P, colour, d, m, blockIdx, gridDim);
}

// ---- CSR: one thread per site of the colour -------------------------------------------------
template <bool DIAG>
__global__ void __launch_bounds__(256)
k_sweep_csr(float* sx, float* sy, float* sz, CsrDev g, uint32_t list_begin, uint32_t list_count,
            SweepParams P, Diag d) {
  resolve_sweep(P);
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
  const bool acc = attempt(i + g.site_base, P, K, ex, ey, ez, hx, hy, hz, ox, oy, oz);
  if (acc) { sx[i] = ox; sy[i] = oy; sz[i] = oz; }
  if (DIAG) {
    if (d.accept) d.accept[i] = acc;
    if (d.n_accept) {   // one atomic per warp (some lanes of the last warp have left)
      const unsigned live = __activemask(), votes = __ballot_sync(live, acc);
      if (votes && (threadIdx.x & 31) == (unsigned)(__ffs(live) - 1)) atomicAdd(d.n_accept, (unsigned long long)__popc(votes));
    }
  }
}

// ---- the paper's own update scheme, emulated (context for BASELINE.md, not the product path) -----------------
// [P:30-32]: "each GPU block handles a part of that array ... N_b blocks are called to perform a spin update in parallel.
// Each block handles n spins, and within each block one of those spins is selected at random to be updated at every step",
// the spins being read from and written to global memory while other blocks update theirs: with small n a spin's
// neighbours change under the energy calculation ("loss of continuity").  Here one THREAD plays one of the paper's
// blocks: it owns the n consecutive sites [t n, (t+1) n) of the linearised (canonical) array, draws one of them, runs rule
// (ii)-(iii) on it against whatever its neighbours hold at that moment, and stores the result.  One launch = one step =
// N / n attempts; one MCS = n steps.  Racy by construction and not reproducible bit for bit: only its statistics and its
// rate are meaningful.  Random numbers: Philox(counter = (t, 2, step), key = seed) picks the site, (site, 3, step) feeds the attempt.
template <int ANISO>
__global__ void __launch_bounds__(256)
k_paper_step(float* s, ScLayout L, SweepParams P, uint32_t n_per_block, uint32_t n_blocks, unsigned long long* n_accept) {
  const uint32_t t = blockIdx.x * blockDim.x + threadIdx.x;
  bool acc = false;
  if (t < n_blocks) {
    const Rand4 pick = philox4x32_10(t, 2u, P.sweep_lo, P.sweep_hi, P.seed_lo, P.seed_hi);
    const uint32_t id = t * n_per_block + pick.r0 % n_per_block;
    const uint32_t Lx = (uint32_t)L.Lx, Ly = (uint32_t)L.Ly, Lz = (uint32_t)L.Lz, H = (uint32_t)L.H;
    const uint32_t x = id % Lx, yz = id / Lx, y = yz % Ly, z = yz / Ly;
    const uint32_t c = (x + y + z) & 1u;
    auto at = [&](uint32_t xx, uint32_t yy, uint32_t zz, uint32_t cc) { return cc * L.half + (zz * Ly + yy) * H + (xx >> 1); };
    const uint32_t m = at(x, y, z, c), o = 1u - c;
    const uint32_t nb[6] = {at(x ? x - 1 : Lx - 1, y, z, o), at(x + 1 < Lx ? x + 1 : 0, y, z, o), at(x, y ? y - 1 : Ly - 1, z, o),
                            at(x, y + 1 < Ly ? y + 1 : 0, z, o), at(x, y, z ? z - 1 : Lz - 1, o), at(x, y, z + 1 < Lz ? z + 1 : 0, o)};
    const size_t n = L.n;
    const volatile float* v = s;       // whatever the other "blocks" have stored by now
    float hx = 0.0f, hy = 0.0f, hz = 0.0f;
#pragma unroll
    for (int k = 0; k < 6; ++k) { hx = __fadd_rn(hx, v[nb[k]]); hy = __fadd_rn(hy, v[n + nb[k]]); hz = __fadd_rn(hz, v[2 * n + nb[k]]); }
    float sx = v[m], sy = v[n + m], sz = v[2 * n + m];
    const Rand4 r = philox4x32_10(id, 3u, P.sweep_lo, P.sweep_hi, P.seed_lo, P.seed_hi);
    float nx, ny, nz;
    sphere(r.r0, r.r1, nx, ny, nz);
    const float dH = delta_h_t<ANISO>(sx, sy, sz, nx, ny, nz, hx, hy, hz, P.J, P.K, P.ex, P.ey, P.ez);
    acc = metropolis_accept(dH, P.beta, r.r2);
    if (acc) { s[m] = nx; s[n + m] = ny; s[2 * n + m] = nz; }
  }
  if (n_accept) {
    const unsigned votes = __ballot_sync(0xffffffffu, acc);
    if (votes && (threadIdx.x & 31) == 0) atomicAdd(n_accept, (unsigned long long)__popc(votes));
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
  for (unsigned long long m64 = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; m64 < L.n; m64 += (unsigned long long)gridDim.x * blockDim.x) {
    const uint32_t m = (uint32_t)m64;   // 64-bit loop index: a 32-bit one wraps below n when n is close to 2^32
    const Rand4 r = philox4x32_10(sc_canonical(L, m) + L.site_base, 1u, 0u, 0u, seed_lo, seed_hi);
    float x, y, z;
    sphere(r.r0, r.r1, x, y, z);
    sx[m] = x; sy[m] = y; sz[m] = z;
  }
}

__global__ void k_init_random_flat(float* sx, float* sy, float* sz, uint32_t n, uint32_t seed_lo, uint32_t seed_hi, uint32_t site_base) {
  for (unsigned long long m64 = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; m64 < n; m64 += (unsigned long long)gridDim.x * blockDim.x) {
    const uint32_t m = (uint32_t)m64;   // 64-bit loop index: a 32-bit one wraps below n when n is close to 2^32
    const Rand4 r = philox4x32_10(m + site_base, 1u, 0u, 0u, seed_lo, seed_hi);
    float x, y, z;
    sphere(r.r0, r.r1, x, y, z);
    sx[m] = x; sy[m] = y; sz[m] = z;
  }
}

// exchange step of table parts (CSR engine: three planes): the spins of the listed local sites <-> packed (x, y, z, 0) records
__global__ void k_part_move_flat(float* sx, float* sy, float* sz, const int32_t* __restrict__ ids, uint32_t count, float4* packed, bool gather) {
  for (unsigned long long k = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; k < count; k += (unsigned long long)gridDim.x * blockDim.x) {
    const int32_t i = ids[k];
    if (gather) packed[k] = make_float4(sx[i], sy[i], sz[i], 0.0f);
    else { const float4 v = packed[k]; sx[i] = v.x; sy[i] = v.y; sz[i] = v.z; }
  }
}

__global__ void k_fill(float* sx, float* sy, float* sz, uint32_t n, float x, float y, float z) {
  for (unsigned long long m64 = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; m64 < n; m64 += (unsigned long long)gridDim.x * blockDim.x) {
    const uint32_t m = (uint32_t)m64;   // 64-bit loop index: a 32-bit one wraps below n when n is close to 2^32
    sx[m] = x; sy[m] = y; sz[m] = z;
  }
}

// dst[m] = src[canonical(m)] (to_internal) or dst[canonical(m)] = src[m]
__global__ void k_sc_permute(float* dst, const float* src, ScLayout L, bool to_internal) {
  for (unsigned long long m64 = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; m64 < L.n; m64 += (unsigned long long)gridDim.x * blockDim.x) {
    const uint32_t m = (uint32_t)m64;   // 64-bit loop index: a 32-bit one wraps below n when n is close to 2^32
    const uint32_t id = sc_canonical(L, m);
    if (to_internal) dst[m] = src[id]; else dst[id] = src[m];
  }
}

// ---- measurement --------------------------------------------------------------------------------
// fixed-order final sum of the block partials by one block (fixed for a given block size)
__device__ __forceinline__ void reduce_final_block(const double* partials, int n_blocks, double* out) {
  // any block size: threads beyond 256 stay out, missing ones leave zeros
  double a[4] = {0, 0, 0, 0};
  const int nt = blockDim.x < 256 ? blockDim.x : 256;
  if ((int)threadIdx.x < nt)
    for (int b = threadIdx.x; b < n_blocks; b += nt)
      for (int q = 0; q < 4; ++q) a[q] += partials[b * 4 + q];
  __shared__ double sh[4][256];
  __syncthreads();
  for (int k = threadIdx.x; k < 256; k += blockDim.x)
    for (int q = 0; q < 4; ++q) sh[q][k] = 0.0;
  __syncthreads();
  if ((int)threadIdx.x < nt)
    for (int q = 0; q < 4; ++q) sh[q][threadIdx.x] = a[q];
  __syncthreads();
  for (int s = 128; s > 0; s >>= 1) {
    if ((int)threadIdx.x < s)
      for (int q = 0; q < 4; ++q) sh[q][threadIdx.x] += sh[q][threadIdx.x + s];
    __syncthreads();
  }
  if (threadIdx.x < 4) out[threadIdx.x] = sh[threadIdx.x][0];
}

__global__ void k_set_counter(unsigned long long* counter, unsigned long long value, bool add) {
  *counter = add ? *counter + value : value;
}

__global__ void __launch_bounds__(256) k_reduce_final(const double* partials, int n_blocks, double* out) {
  reduce_final_block(partials, n_blocks, out);
}

// the same for replayed launches: entry *idx of a series (4 doubles per entry), then *idx advances
__global__ void __launch_bounds__(256) k_reduce_final_series(const double* partials, int n_blocks, double* series,
                                                             unsigned long long* idx) {
  const unsigned long long i = *idx;
  reduce_final_block(partials, n_blocks, series + 4 * i);
  __syncthreads();
  if (threadIdx.x == 0) *idx = i + 1;
}

// ---- persistent multi-sweep kernel for lattices whose colour pass is shorter than a kernel launch ----------
// One cooperative launch runs n_sweeps sweeps: every block walks the virtual blocks of a colour pass, then the
// whole grid meets at a barrier (cooperative groups) before the next colour.  Same arithmetic, same tiles, same
// bits as the one-launch-per-colour path; what it removes is the launch gap (5-6 us per colour on B200, against
// 1-2 us of work for L <= 128).  Measurement (fused, section 6.5): with series != nullptr EVERY sweep is measured
// and (sum S, E) of sweep s goes to series[4 s ..]; else with final_out != nullptr only the last sweep is.
// Block 0 sums the block partials of sweep s while the grid already runs colour 0 of sweep s+1, so the partials
// are double-buffered by sweep parity (2 x 2 x total x 4 doubles).
// ONE: the whole colour pass fits one block of up to 1024 threads (N <= 8192): a single block on a single SM, the
// barrier is __syncthreads and the 12 N bytes of state stay in that SM's L1.  A grid of such blocks runs independent
// REPLICAS of the lattice, one per block (state of replica r at s + 3 N r, Philox key seed + r, its own beta, its own
// partials / series / final_out): many temperatures or seeds of a small lattice per launch.
template <int ANISO, bool ONE>
__global__ void __launch_bounds__(ONE ? 1024 : 256, ONE ? 1 : 3)
k_sweeps_sc_coop(float* s, ScLayout L, ScTile t, SweepParams P, unsigned long long sweep0, int n_sweeps, uint3 nblk,
                 double* partials, double* series, double* final_out, const float* betas, unsigned long long series_stride,
                 unsigned long long* n_accept) {
  cooperative_groups::grid_group grid = cooperative_groups::this_grid();
  const size_t n = L.n;
  const uint32_t total = nblk.x * nblk.y * nblk.z;
  const Diag d{nullptr, nullptr};
  if (ONE) {
    t.LIN = -1;
    const unsigned long long r = blockIdx.x;
    const unsigned long long seed = (((unsigned long long)P.seed_hi << 32) | P.seed_lo) + r;
    P.seed_lo = (uint32_t)seed; P.seed_hi = (uint32_t)(seed >> 32);
    if (betas) P.beta = betas[r];
    s += 3 * n * r;
    partials += 16 * r;
    if (series) series += series_stride * r;
    if (final_out) final_out += 4 * r;
  }
  for (int sw = 0; sw < n_sweeps; ++sw) {
    const unsigned long long sc = sweep0 + (unsigned long long)sw;
    P.sweep_lo = (uint32_t)sc; P.sweep_hi = (uint32_t)(sc >> 32);
    const bool meas = series != nullptr || (final_out != nullptr && sw == n_sweeps - 1);
    double* part = partials + (size_t)(sw & 1) * 2 * total * 4;
    for (int colour = 0; colour < 2; ++colour) {
      float* a = s + (size_t)colour * L.half;
      const float* b = s + (size_t)(1 - colour) * L.half;
      for (uint32_t v = ONE ? 0u : blockIdx.x; v < total; v += ONE ? 1u : gridDim.x) {
        const uint3 bid = make_uint3(v % nblk.x, (v / nblk.x) % nblk.y, v / (nblk.x * nblk.y));
        if (meas) {
          const Meas mc{part + (size_t)colour * total * 4, colour == 1 ? 2 : 1, n_accept};
          sc_pass<4, ANISO, false, 0, true, true>(a, a + n, a + 2 * n, b, b + n, b + 2 * n, L, t, P, colour, d, mc, bid, nblk);
        } else {
          sc_pass<4, ANISO, false, 0, false, true>(a, a + n, a + 2 * n, b, b + n, b + 2 * n, L, t, P, colour, d, Meas{nullptr, 0, nullptr}, bid, nblk);
        }
      }
      if (ONE) __syncthreads(); else grid.sync();
    }
    if (ONE) {   // two partials (one per colour), already behind the colour step's barrier: same sum, no tree
      if (meas && threadIdx.x < 4) (series ? series + 4 * (size_t)sw : final_out)[threadIdx.x] = part[threadIdx.x] + part[4 + threadIdx.x];
    } else if (meas && blockIdx.x == 0) {
      reduce_final_block(part, 2 * (int)total, series ? series + 4 * (size_t)sw : final_out);
    }
  }
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
    if (L.ghost && (z == 0 || z == L.Lz - 1)) continue;   // a slab sums its own planes only
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
  block_reduce4(mx, my, mz, en, partials + (size_t)blockIdx.x * 4);
}

__global__ void __launch_bounds__(256)
k_measure_csr(const float* __restrict__ sx, const float* __restrict__ sy, const float* __restrict__ sz,
              CsrDev g, SweepParams P, double* partials) {
  double mx = 0, my = 0, mz = 0, en = 0;
  for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < g.n_own; i += gridDim.x * blockDim.x) {   // (ghost sites of a part are not measured)
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
  block_reduce4(mx, my, mz, en, partials + (size_t)blockIdx.x * 4);
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

cudaError_t launch_init_random_flat(cudaStream_t st, float* s, uint32_t n, uint32_t seed_lo, uint32_t seed_hi, uint32_t site_base) {
  k_init_random_flat<<<grid_for(n, 256, 148 * 16), 256, 0, st>>>(s, s + n, s + 2 * (size_t)n, n, seed_lo, seed_hi, site_base);
  return cudaGetLastError();
}

cudaError_t launch_part_move_flat(cudaStream_t st, float* s, uint32_t n, const int32_t* ids, uint32_t count, float* packed, bool gather) {
  if (count == 0) return cudaSuccess;
  k_part_move_flat<<<grid_for(count, 256, 148 * 8), 256, 0, st>>>(s, s + n, s + 2 * (size_t)n, ids, count, reinterpret_cast<float4*>(packed), gather);
  return cudaGetLastError();
}

cudaError_t launch_fill(cudaStream_t st, float* s, uint32_t n, float x, float y, float z) {
  k_fill<<<grid_for(n, 256, 148 * 16), 256, 0, st>>>(s, s + n, s + 2 * (size_t)n, n, x, y, z);
  return cudaGetLastError();
}

inline int aniso_case(const SweepParams& p);

cudaError_t launch_paper_step(cudaStream_t st, float* s, ScLayout L, SweepParams p, uint32_t n_per_block, unsigned long long* n_accept) {
  const uint32_t n_blocks = L.n / n_per_block;
  const unsigned grid = (n_blocks + 255u) / 256u;
  switch (aniso_case(p)) {
    case ANISO_NONE: k_paper_step<ANISO_NONE><<<grid, 256, 0, st>>>(s, L, p, n_per_block, n_blocks, n_accept); break;
    case ANISO_Z: k_paper_step<ANISO_Z><<<grid, 256, 0, st>>>(s, L, p, n_per_block, n_blocks, n_accept); break;
    default: k_paper_step<ANISO_GENERAL><<<grid, 256, 0, st>>>(s, L, p, n_per_block, n_blocks, n_accept); break;
  }
  return cudaGetLastError();
}

cudaError_t launch_sc_permute(cudaStream_t st, float* dst, const float* src, ScLayout L, bool to_internal) {
  k_sc_permute<<<grid_for(L.n, 256, 148 * 16), 256, 0, st>>>(dst, src, L, to_internal);
  return cudaGetLastError();
}

inline int aniso_case(const SweepParams& p) {
  return (p.K == 0.0f) ? ANISO_NONE : ((p.ex == 0.0f && p.ey == 0.0f && p.ez == 1.0f) ? ANISO_Z : ANISO_GENERAL);
}

// launch shape of k_sweep_sc for a tile
static void sc_launch_shape(const ScLayout& L, const ScTile& t, int V, dim3& grid, int& threads) {
  const int HV = L.H / V;
  threads = t.LIN ? t.LIN : t.JX * t.TY;
  grid = dim3((HV + t.JX - 1) / t.JX, (L.Ly + t.TY - 1) / t.TY, (L.Lz + t.ZT - 1) / t.ZT);
  if (t.LIN) grid = dim3((unsigned)(((long long)HV * L.Ly + threads - 1) / threads), 1, (L.Lz + t.ZT - 1) / t.ZT);
}

int sc_fused_blocks(const ScLayout& L, const ScTile& t) {
  if (t.V != 4) return 0;                    // the fused measurement is built for the tuned vector width
  dim3 grid; int threads;
  sc_launch_shape(L, t, 4, grid, threads);
  const long long blocks = (long long)grid.x * grid.y * grid.z;
  return blocks <= kFusedBlocksMax ? (int)blocks : 0;
}

template <int V, int ANISO, bool DIAG>
static cudaError_t sweep_sc_impl(cudaStream_t st, float* s, ScLayout L, ScTile t, SweepParams p, int colour, Diag d, Meas m) {
  int threads = t.LIN ? t.LIN : t.JX * t.TY;
  auto kern = k_sweep_sc<V, ANISO, DIAG, 0>;
  constexpr bool TUNED = !DIAG && V == 4;   // the tuned configuration carries the prefetch, big-block and fused-measurement variants
  constexpr int P1 = TUNED ? 1 : 0, B512 = TUNED ? 512 : 256, B1024 = TUNED ? 1024 : 256;
  if (m.mode != 0 && !TUNED) return cudaErrorInvalidValue;
  if (L.ghost) {   // slab contexts: one variant (blocks of up to 256 threads, no fused measurement, no recording)
    if (m.mode != 0 || DIAG) return cudaErrorInvalidValue;
    kern = k_sweep_sc<V, ANISO, DIAG, P1, 256, false, true>;
    if (threads > 256) {
      if (t.JX > 256) t.JX = 256;
      t.TY = 256 / t.JX;
      if (t.LIN > 256) t.LIN = 256;
    }
  } else if (TUNED) {
    if (m.mode != 0) {
      if (threads > 512) kern = k_sweep_sc<V, ANISO, DIAG, P1, B1024, TUNED>;
      else if (threads > 256) kern = k_sweep_sc<V, ANISO, DIAG, P1, B512, TUNED>;
      else kern = k_sweep_sc<V, ANISO, DIAG, P1, 256, TUNED>;
    } else if (threads > 512) kern = t.PF ? k_sweep_sc<V, ANISO, DIAG, P1, B1024> : k_sweep_sc<V, ANISO, DIAG, 0, B1024>;
    else if (threads > 256) kern = t.PF ? k_sweep_sc<V, ANISO, DIAG, P1, B512> : k_sweep_sc<V, ANISO, DIAG, 0, B512>;
    else switch (t.PF) {
      case 1: kern = k_sweep_sc<V, ANISO, DIAG, P1>; break;
      case 2: kern = k_sweep_sc<V, ANISO, DIAG, TUNED ? 2 : 0>; break;
      case 3: kern = k_sweep_sc<V, ANISO, DIAG, TUNED ? 3 : 0>; break;
      default: break;
    }
  } else if (threads > 256) {   // the other variants are built for blocks of up to 256 threads: shrink the tile
    if (t.JX > 256) t.JX = 256;
    t.TY = 256 / t.JX;
  }
  const size_t n = L.n;
  float* a = s + (size_t)colour * L.half;
  const float* b = s + (size_t)(1 - colour) * L.half;
  dim3 grid;
  sc_launch_shape(L, t, V, grid, threads);
  return launch_colour_kernel(kern, grid, dim3(threads), 0, st, p.pdl != 0, a, a + n, a + 2 * n, b, b + n, b + 2 * n, L, t, p, colour, d, m);
}

template <int V, bool DIAG>
static cudaError_t sweep_sc_aniso(cudaStream_t st, float* s, ScLayout L, ScTile t, SweepParams p, int colour, Diag d, Meas m) {
  switch (aniso_case(p)) {
    case ANISO_NONE: return sweep_sc_impl<V, ANISO_NONE, DIAG>(st, s, L, t, p, colour, d, m);
    case ANISO_Z: return sweep_sc_impl<V, ANISO_Z, DIAG>(st, s, L, t, p, colour, d, m);
    default: return sweep_sc_impl<V, ANISO_GENERAL, DIAG>(st, s, L, t, p, colour, d, m);
  }
}

cudaError_t launch_sweep_sc(cudaStream_t st, float* s, ScLayout L, ScTile t, SweepParams p, int colour, Diag d, Meas m) {
  const bool diag = d.accept || d.n_accept;
  switch (t.V) {
    case 4: return diag ? sweep_sc_aniso<4, true>(st, s, L, t, p, colour, d, m) : sweep_sc_aniso<4, false>(st, s, L, t, p, colour, d, m);
    case 2: return diag ? sweep_sc_aniso<2, true>(st, s, L, t, p, colour, d, m) : sweep_sc_aniso<2, false>(st, s, L, t, p, colour, d, m);
    default: return diag ? sweep_sc_aniso<1, true>(st, s, L, t, p, colour, d, m) : sweep_sc_aniso<1, false>(st, s, L, t, p, colour, d, m);
  }
}

// threads of the one-block path if a whole colour pass fits one block (V = 4, N/8 <= 1024 threads), else 0
int sc_one_block_threads(const ScLayout& L) {
  if (L.H % 4 != 0) return 0;
  const long long slots = (long long)(L.H / 4) * L.Ly * L.Lz;
  return slots <= 1024 ? (int)((slots + 31) / 32 * 32) : 0;
}

// persistent cooperative path: virtual blocks of a colour pass (0 = not available for this tile)
int sc_coop_blocks(const ScLayout& L, const ScTile& t) {
  if (t.V != 4 || (t.LIN ? t.LIN : t.JX * t.TY) > 256) return 0;
  dim3 grid; int threads;
  sc_launch_shape(L, t, 4, grid, threads);
  const long long blocks = (long long)grid.x * grid.y * grid.z;
  return blocks <= kFusedBlocksMax / 2 ? (int)blocks : 0;
}

cudaError_t launch_sweeps_sc_coop(cudaStream_t st, float* s, ScLayout L, ScTile t, SweepParams p, uint64_t sweep0, int n_sweeps,
                                  bool one_block, double* partials, double* series, double* final_out,
                                  int n_replicas, const float* betas, uint64_t series_stride, unsigned long long* n_accept) {
  const int aniso = aniso_case(p);
  if (one_block) {
    const int threads = sc_one_block_threads(L);
    if (!threads || n_replicas < 1) return cudaErrorInvalidValue;
    const uint3 nblk = make_uint3(1, 1, 1);
    const unsigned long long stride = series_stride;
    switch (aniso) {
      case ANISO_NONE: k_sweeps_sc_coop<ANISO_NONE, true><<<n_replicas, threads, 0, st>>>(s, L, t, p, sweep0, n_sweeps, nblk, partials, series, final_out, betas, stride, n_accept); break;
      case ANISO_Z: k_sweeps_sc_coop<ANISO_Z, true><<<n_replicas, threads, 0, st>>>(s, L, t, p, sweep0, n_sweeps, nblk, partials, series, final_out, betas, stride, n_accept); break;
      default: k_sweeps_sc_coop<ANISO_GENERAL, true><<<n_replicas, threads, 0, st>>>(s, L, t, p, sweep0, n_sweeps, nblk, partials, series, final_out, betas, stride, n_accept); break;
    }
    return cudaGetLastError();
  }
  dim3 vgrid; int threads;
  sc_launch_shape(L, t, 4, vgrid, threads);
  void (*kern)(float*, ScLayout, ScTile, SweepParams, unsigned long long, int, uint3, double*, double*, double*, const float*, unsigned long long, unsigned long long*);
  switch (aniso) {
    case ANISO_NONE: kern = k_sweeps_sc_coop<ANISO_NONE, false>; break;
    case ANISO_Z: kern = k_sweeps_sc_coop<ANISO_Z, false>; break;
    default: kern = k_sweeps_sc_coop<ANISO_GENERAL, false>; break;
  }
  int dev = 0, sms = 0, per_sm = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, threads, 0);
  if (e != cudaSuccess) return e;
  if (per_sm < 1) return cudaErrorLaunchOutOfResources;
  const long long total = (long long)vgrid.x * vgrid.y * vgrid.z;
  const long long resident = (long long)per_sm * sms;
  const unsigned grid = (unsigned)(total < resident ? total : resident);
  uint3 nblk = make_uint3(vgrid.x, vgrid.y, vgrid.z);
  unsigned long long s0 = sweep0;
  const float* no_betas = nullptr;
  unsigned long long no_stride = 0;
  void* args[] = {&s, &L, &t, &p, &s0, &n_sweeps, &nblk, &partials, &series, &final_out, &no_betas, &no_stride, &n_accept};
  return cudaLaunchCooperativeKernel((const void*)kern, dim3(grid), dim3(threads), args, 0, st);
}

cudaError_t launch_sweep_csr(cudaStream_t st, float* s, CsrDev g, uint32_t list_begin, uint32_t list_count,
                             SweepParams p, int block, Diag d) {
  if (list_count == 0) return cudaSuccess;
  const size_t n = g.n;
  const int grid = (int)((list_count + block - 1) / block);
  if (d.accept || d.n_accept)
    return launch_colour_kernel(k_sweep_csr<true>, dim3(grid), dim3(block), 0, st, p.pdl != 0, s, s + n, s + 2 * n, g, list_begin, list_count, p, d);
  return launch_colour_kernel(k_sweep_csr<false>, dim3(grid), dim3(block), 0, st, p.pdl != 0, s, s + n, s + 2 * n, g, list_begin, list_count, p, d);
}

cudaError_t launch_set_counter(cudaStream_t st, unsigned long long* counter, unsigned long long value, bool add) {
  k_set_counter<<<1, 1, 0, st>>>(counter, value, add);
  return cudaGetLastError();
}

cudaError_t launch_reduce_final_series(cudaStream_t st, const double* partials, int n_blocks, double* series,
                                       unsigned long long* idx) {
  k_reduce_final_series<<<1, 256, 0, st>>>(partials, n_blocks, series, idx);
  return cudaGetLastError();
}

cudaError_t launch_reduce_final(cudaStream_t st, const double* partials, int n_blocks, double* out) {
  k_reduce_final<<<1, 256, 0, st>>>(partials, n_blocks, out);
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
