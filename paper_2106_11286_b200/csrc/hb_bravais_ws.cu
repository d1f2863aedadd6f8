// hb_bravais_ws.cu -- bcc / fcc colour passes, warp-specialised and persistent: the producer-warp /
// bulk-copy treatment of hb_sc_ws.cu for the lattices with a basis.
//
// The direct kernel (hb_bravais.cu) reads every neighbour row through L1: 24 (bcc) or 36 (fcc) vector loads per thread and
// plane that miss half of the time, one short-lived block per tile, several waves per launch.  Here
//   * one PRODUCER warp per CTA streams, with 1-D bulk asynchronous copies (cp.async.bulk, the TMA engine) completing on
//     mbarriers, "groups" into a ring in shared memory: group g of a tile = for every OTHER sublattice the rows
//     y0+dylo .. y0+TY+dylo of plane z0+dzlo+g, three components each (the neighbours of a sublattice lie in a window of two
//     rows and two planes: hb_bravais_geo.cuh), so a plane step reads groups g and g+1 and a group serves two steps;
//   * the CONSUMER warps read all 8 / 12 neighbour vectors with LDS at compile-time offsets (the geometry is a template
//     constant, the periodic wrap in x is an index inside the staged row), sum them in the contract's order, run the attempt
//     arithmetic of hb_device.cuh, load and store their own spins themselves;
//   * CTAs are persistent and take tiles (TY rows x a chunk of planes) from a device counter.
// FUSED: all colour passes of several sweeps in ONE launch, ordered in rounds with progress words between consecutive
// passes, exactly as in hb_sc_ws.cu (pass p = sweep p / NB, colour p % NB; a tile of pass p waits for the chunks k, k+1, k+2
// of pass p-1, which in turn waited for pass p-2, ...).  For lattices whose colour pass is shorter than a kernel launch
// (c2: 262,144 updates, 4 us) this takes the launch boundary out of the sweep altogether.
//
// Same arithmetic, same order of the neighbour sum, same bits as k_sweep_bravais.
#include "hb_device.cuh"
#include "hb_internal.h"
#include "hb_ws.cuh"
#include "hb_bravais_geo.cuh"

namespace hb {

namespace {

template <int KIND, int TY, int ROWB, int kNB>
struct BwSmem {
  static constexpr int NO = Geo<KIND>::NB - 1;                       // other sublattices
  static constexpr uint32_t COMP_B = (uint32_t)(TY + 1) * ROWB;      // one component of one sublattice in a group
  static constexpr uint32_t GROUP_B = (uint32_t)NO * 3u * COMP_B;
  static constexpr uint32_t OFF_BAR = kNB * GROUP_B;                 // full[kNB], empty[kNB]
  static constexpr uint32_t OFF_TILE = OFF_BAR + 16u * kNB;          // info[kNB]: x = tile (-1: no more), y = pass, z = chunk, w = tile in y
  static constexpr uint32_t BYTES = OFF_TILE + 16u * kNB;
};

template <int V, int TY, int ROWB>
__host__ __device__ constexpr int bw_max_threads() {
  const int t = 32 + 32 * ((TY * (ROWB / (4 * V)) + 31) / 32);
  return t > 1024 ? 1024 : t;
}

// ---- producer: one warp ------------------------------------------------------------------------------------------------
template <int KIND, int TY, int ROWB, int kNB>
__device__ __forceinline__ void bw_producer(const float* s, const BrLayout& L, const WsTiles& w,
                                            unsigned char* smem, uint32_t sbase) {
  using S = BwSmem<KIND, TY, ROWB, kNB>;
  constexpr int NB = Geo<KIND>::NB;
  const uint32_t lane = threadIdx.x;
  const uint32_t row_bytes = (uint32_t)L.Lx * 4u;
  const size_t n = L.n;
  const uint32_t fullB = sbase + S::OFF_BAR, emptyB = fullB + 8u * kNB;
  RingPos<kNB> rp;
  const int32_t n_tiles = w.n_ty * w.n_zc * w.passes;
  volatile int4* info = reinterpret_cast<volatile int4*>(smem + S::OFF_TILE);
  for (;;) {
    int32_t tile = 0;
    if (lane == 0) tile = (int32_t)atomicAdd(w.sched, 1u);
    tile = __shfl_sync(0xffffffffu, tile, 0);
    if (tile >= n_tiles) {
      mbar_wait_backoff(emptyB + 8u * rp.slot, rp.par ^ 1u);
      if (lane == 0) { info[rp.slot].x = -1; mbar_arrive(fullB + 8u * rp.slot); }
      break;
    }
    // every launch is a sequence of passes: pass p updates colour (first + p) mod NB (one pass: a plain colour launch)
    const FusedTile t = fused_decode(tile, w);
    const int32_t ty = t.ty, zc = t.zc, pass = t.p, b = (w.first + t.p) % NB;
    if (t.p > 0) {   // the chunks of the previous pass this tile reads, and whose readers must be done before it writes
      if (lane < 3) {
        const uint32_t* d = w.done + (size_t)(t.p - 1) * w.n_zc + (t.k + (int32_t)lane) % w.n_zc;
        const uint32_t all = (uint32_t)w.n_ty * ((blockDim.x >> 5) - 1u);
        while (ld_acquire_gpu(d) < all) __nanosleep(128);
      }
      __syncwarp();
      asm volatile("fence.proxy.async;" ::: "memory");   // the bulk copies below read what other CTAs stored (generic proxy)
    }
    const int32_t dylo = window_lo<KIND>(b, 1), dzlo = window_lo<KIND>(b, 2);
    const int32_t y0 = ty * TY, ny = min(TY, L.Ly - y0);
    const int32_t z0 = (int32_t)(((int64_t)zc * L.Lz) / w.n_zc), nz = (int32_t)(((int64_t)(zc + 1) * L.Lz) / w.n_zc) - z0;
    const uint32_t rows = (uint32_t)(ny + 1), n_copies = (uint32_t)S::NO * 3u * rows;
    for (int32_t g = 0; g <= nz; ++g) {
      int32_t zz = z0 + dzlo + g;
      zz = zz < 0 ? zz + L.Lz : (zz >= L.Lz ? zz - L.Lz : zz);
      const uint32_t slot = rp.slot;
      mbar_wait_backoff(emptyB + 8u * slot, rp.par ^ 1u);
      if (lane == 0) {
        info[slot].x = tile; info[slot].y = pass; info[slot].z = zc; info[slot].w = ty;
        mbar_expect_tx(fullB + 8u * slot, n_copies * row_bytes);
      }
      __syncwarp();
      for (uint32_t q = lane; q < n_copies; q += 32) {
        const uint32_t oc = q / rows, r = q - oc * rows;          // oc = other-sublattice index * 3 + component
        const uint32_t o = oc / 3u, comp = oc - 3u * o;
        const uint32_t nb = o < (uint32_t)b ? o : o + 1u;
        int32_t yy = y0 + dylo + (int32_t)r;
        yy = yy < 0 ? yy + L.Ly : (yy >= L.Ly ? yy - L.Ly : yy);
        const float* src = s + comp * n + (size_t)nb * L.nc + ((size_t)zz * L.Ly + yy) * L.Lx;
        bulk_g2s(sbase + slot * S::GROUP_B + oc * S::COMP_B + r * ROWB, src, row_bytes, fullB + 8u * slot);
      }
      rp.next();
    }
  }
}

// ---- consumers ---------------------------------------------------------------------------------------------------------
// what a consumer thread knows about its V cells of row r of the tile: byte offsets inside one staged row
struct BwWhere {
  uint32_t v0;        // its V-vector
  uint32_t lo, hi;    // the cell left of it and the cell right of its last one (periodic in x)
};

template <int V> __device__ __forceinline__ Vec<V> lds_vec(const unsigned char* p);
template <> __device__ __forceinline__ Vec<4> lds_vec<4>(const unsigned char* p) {
  const float4 t = *reinterpret_cast<const float4*>(p);
  return Vec<4>{{t.x, t.y, t.z, t.w}};
}
template <> __device__ __forceinline__ Vec<2> lds_vec<2>(const unsigned char* p) {
  const float2 t = *reinterpret_cast<const float2*>(p);
  return Vec<2>{{t.x, t.y}};
}

// the V cells shifted by dx in {-1, 0, +1} along the staged row
template <int V>
__device__ __forceinline__ Vec<V> lds_shifted(const unsigned char* row, const BwWhere& w, int dx) {
  const Vec<V> c = lds_vec<V>(row + w.v0);
  if (dx == 0) return c;
  Vec<V> t;
  if (dx < 0) {
    t.v[0] = *reinterpret_cast<const float*>(row + w.lo);
#pragma unroll
    for (int k = 1; k < V; ++k) t.v[k] = c.v[k - 1];
  } else {
#pragma unroll
    for (int k = 0; k + 1 < V; ++k) t.v[k] = c.v[k + 1];
    t.v[V - 1] = *reinterpret_cast<const float*>(row + w.hi);
  }
  return t;
}

template <int V>
__device__ __forceinline__ Vec<V> bw_vadd(const Vec<V>& a, const Vec<V>& b) {
  Vec<V> r;
#pragma unroll
  for (int k = 0; k + 1 < V; k += 2) {
    const f2 s = add2(make_float2(a.v[k], a.v[k + 1]), make_float2(b.v[k], b.v[k + 1]));
    r.v[k] = s.x; r.v[k + 1] = s.y;
  }
  return r;
}

// h = sum over the Z neighbours of sublattice B in contract order, starting from the first one (as k_sweep_bravais);
// LOW: only the neighbours on lower sublattices, starting from zero (the bonds the fused measurement charges here).
// G[0], G[1]: the two staged groups (planes z+dzlo, z+dzlo+1); row0 = byte offset of the thread's row r (window row 0)
template <int KIND, int B, int V, int TY, int ROWB, int kNB, bool LOW, int K = 0>
__device__ __forceinline__ void bw_field(const unsigned char* const G[2], uint32_t row0, const BwWhere& w,
                                         Vec<V>& hx, Vec<V>& hy, Vec<V>& hz) {
  using S = BwSmem<KIND, TY, ROWB, kNB>;
  if constexpr (LOW && K == 0) {
#pragma unroll
    for (int k = 0; k < V; ++k) { hx.v[k] = 0.0f; hy.v[k] = 0.0f; hz.v[k] = 0.0f; }
  }
  if constexpr (K < Geo<KIND>::Z) {
    constexpr Nbr g = Geo<KIND>::nbr(B, K);
    if constexpr (!LOW || g.nb < B) {
      constexpr int o = g.nb < B ? g.nb : g.nb - 1;
      constexpr int wr = g.dy - window_lo<KIND>(B, 1), wz = g.dz - window_lo<KIND>(B, 2);
      const unsigned char* row = G[wz] + (uint32_t)(o * 3) * S::COMP_B + (uint32_t)wr * ROWB + row0;
      const Vec<V> tx = lds_shifted<V>(row, w, g.dx);
      const Vec<V> ty = lds_shifted<V>(row + S::COMP_B, w, g.dx);
      const Vec<V> tz = lds_shifted<V>(row + 2u * S::COMP_B, w, g.dx);
      if constexpr (!LOW && K == 0) { hx = tx; hy = ty; hz = tz; }
      else { hx = bw_vadd<V>(hx, tx); hy = bw_vadd<V>(hy, ty); hz = bw_vadd<V>(hz, tz); }
    }
    bw_field<KIND, B, V, TY, ROWB, kNB, LOW, K + 1>(G, row0, w, hx, hy, hz);
  }
}

// what a tile needs from the kernel's frame
struct BwTile {
  int32_t y0, ny, z0, nz;
  uint32_t sweep_lo, sweep_hi;
  int32_t meas;       // the tile's pass carries the fused measurement
};

// FUSED: bump the progress word of the tile this warp finished last (whole warp, converged).  Deferred to just before the
// first stores of the next tile, when the fence no longer waits for the earlier stores (hb_sc_ws.cu, publish).
__device__ __forceinline__ void bw_publish(uint32_t*& pending) {
  __syncwarp();
  if ((threadIdx.x & 31) == 0) {
    asm volatile("fence.proxy.async;" ::: "memory");
    __threadfence();
    atomicAdd(pending, 1u);
  }
  pending = nullptr;
}

// all plane steps of one tile of sublattice B
template <int KIND, int B, int V, int TY, int ROWB, int kNB, int ANISO, bool MEAS>
__device__ __forceinline__ void bw_tile(float* s, const BrLayout& L, const SweepParams& P, const BwTile& t, unsigned char* smem,
                                        uint32_t sbase, RingPos<kNB>& rm, double acc[4], unsigned& n_acc, uint32_t*& pending) {
  using S = BwSmem<KIND, TY, ROWB, kNB>;
  const uint32_t fullB = sbase + S::OFF_BAR, emptyB = fullB + 8u * kNB;
  const int32_t HV = L.Lx / V;
  const int32_t c = (int32_t)threadIdx.x - 32;
  const int32_t r = c / HV, j = c - r * HV, i0 = j * V;
  const bool lane0 = (threadIdx.x & 31) == 0;
  const bool active = r < t.ny;
  BwWhere w;
  w.v0 = (uint32_t)i0 * 4u;
  w.lo = (uint32_t)(i0 == 0 ? L.Lx - 1 : i0 - 1) * 4u;
  w.hi = (uint32_t)(i0 + V >= L.Lx ? i0 + V - L.Lx : i0 + V) * 4u;
  const uint32_t row0 = (uint32_t)r * ROWB;
  const size_t n = L.n, plane = (size_t)L.Ly * L.Lx;
  const int32_t y = t.y0 + r;
  float* gx = s + (size_t)B * L.nc + ((size_t)t.z0 * L.Ly + y) * L.Lx + i0;
  uint32_t site0 = (uint32_t)B * L.nc + (uint32_t)((t.z0 * L.Ly + y) * L.Lx + i0);   // canonical id = b*Nc + cell
  for (int32_t st = 0; st < t.nz; ++st) {
    Vec<V> sx, sy, sz;
    if (active) {
      // an earlier pass of this launch, on any SM, may have written them: read at the L2, never a line kept in this SM's L1
      sx = load_cg<V>(gx); sy = load_cg<V>(gx + n); sz = load_cg<V>(gx + 2 * n);
    }
    RingPos<kNB> rc = rm; rc.next();
    if (st == 0) mbar_wait(fullB + 8u * rm.slot, rm.par);
    mbar_wait(fullB + 8u * rc.slot, rc.par);
    const unsigned char* const G[2] = {smem + rm.slot * S::GROUP_B, smem + rc.slot * S::GROUP_B};
    Vec<V> hx, hy, hz, lx, ly, lz;
    if (active) {
      bw_field<KIND, B, V, TY, ROWB, kNB, false>(G, row0, w, hx, hy, hz);
      if (MEAS && n_low<KIND, B>() != Geo<KIND>::Z && n_low<KIND, B>() != 0) { if (t.meas) bw_field<KIND, B, V, TY, ROWB, kNB, true>(G, row0, w, lx, ly, lz); }
    }
    __syncwarp();
    if (lane0) {   // this warp is done with the older group (after the last plane of the tile: with both)
      mbar_arrive(emptyB + 8u * rm.slot);
      if (st == t.nz - 1) mbar_arrive(emptyB + 8u * rc.slot);
    }
    bool any = false;
    if (active) {
#pragma unroll
      for (int k = 0; k + 1 < V; k += 2) {
        const Rand4 ra = philox4x32_10(site0 + k, 0u, t.sweep_lo, t.sweep_hi, P.seed_lo, P.seed_hi);
        const Rand4 rb = philox4x32_10(site0 + k + 1, 0u, t.sweep_lo, t.sweep_hi, P.seed_lo, P.seed_hi);
        f2 px = make_float2(sx.v[k], sx.v[k + 1]), py = make_float2(sy.v[k], sy.v[k + 1]), pz = make_float2(sz.v[k], sz.v[k + 1]);
        bool acc_a, acc_b;
        attempt2<ANISO>(ra, rb, P.J, P.K, P.beta, P.ex, P.ey, P.ez, make_float2(hx.v[k], hx.v[k + 1]),
                        make_float2(hy.v[k], hy.v[k + 1]), make_float2(hz.v[k], hz.v[k + 1]), px, py, pz, acc_a, acc_b);
        sx.v[k] = px.x; sx.v[k + 1] = px.y; sy.v[k] = py.x; sy.v[k + 1] = py.y; sz.v[k] = pz.x; sz.v[k + 1] = pz.y;
        any |= acc_a | acc_b;
        if (MEAS) n_acc += t.meas ? (unsigned)acc_a + (unsigned)acc_b : 0u;
      }
    }
    if (pending) bw_publish(pending);
    if (active) {
      if (any) {
        store<V>(gx, sx);
        store<V>(gx + n, sy);
        store<V>(gx + 2 * n, sz);
      }
      if (MEAS) {
        if (t.meas) {
          if constexpr (n_low<KIND, B>() == Geo<KIND>::Z) { lx = hx; ly = hy; lz = hz; }   // highest colour: the whole field
          if constexpr (n_low<KIND, B>() == 0) {
#pragma unroll
            for (int k = 0; k < V; ++k) { lx.v[k] = 0.0f; ly.v[k] = 0.0f; lz.v[k] = 0.0f; }
          }
          float mx = 0.0f, my = 0.0f, mz = 0.0f, me = 0.0f;
#pragma unroll
          for (int k = 0; k < V; ++k) {
            mx = __fadd_rn(mx, sx.v[k]); my = __fadd_rn(my, sy.v[k]); mz = __fadd_rn(mz, sz.v[k]);
            const float sl = __fmaf_rn(sz.v[k], lz.v[k], __fmaf_rn(sy.v[k], ly.v[k], __fmul_rn(sx.v[k], lx.v[k])));
            const float a = __fmaf_rn(sz.v[k], P.ez, __fmaf_rn(sy.v[k], P.ey, __fmul_rn(sx.v[k], P.ex)));
            me = __fadd_rn(me, __fmaf_rn(-P.J, sl, __fmul_rn(-P.K, __fmul_rn(a, a))));
          }
          acc[0] += (double)mx; acc[1] += (double)my; acc[2] += (double)mz; acc[3] += (double)me;
        }
      }
    }
    gx += plane;
    site0 += (uint32_t)plane;
    rm.next();
  }
  rm.next();   // the extra group of the tile
}

template <int KIND, int V, int TY, int ROWB, int kNB, int ANISO, bool MEAS>
__device__ __forceinline__ void bw_consumer(float* s, const BrLayout& L, const WsTiles& w, const SweepParams& P, int mode,
                                            unsigned char* smem, uint32_t sbase, double acc[4], unsigned& n_acc) {
  using S = BwSmem<KIND, TY, ROWB, kNB>;
  constexpr int NB = Geo<KIND>::NB;
  const uint32_t fullB = sbase + S::OFF_BAR;
  RingPos<kNB> rm;
  const volatile int4* info = reinterpret_cast<const volatile int4*>(smem + S::OFF_TILE);
  uint32_t* pending = nullptr;
  for (;;) {
    if (pending) {   // deferring is safe once the producer is past the dependencies of the next tile (hb_sc_ws.cu)
      uint32_t staged = 0;
      if ((threadIdx.x & 31) == 0) staged = mbar_test(fullB + 8u * rm.slot, rm.par) ? 1u : 0u;
      if (!__shfl_sync(0xffffffffu, staged, 0)) bw_publish(pending);
    }
    mbar_wait(fullB + 8u * rm.slot, rm.par);
    const int32_t tile = info[rm.slot].x;
    if (tile < 0) { if (pending) bw_publish(pending); break; }
    const int32_t pass = info[rm.slot].y, zc = info[rm.slot].z, ty = info[rm.slot].w;
    const int32_t gp = w.first + pass, b = gp % NB;   // pass p of the launch: colour (first + p) mod NB of sweep (first + p) / NB
    BwTile t;
    const unsigned long long sw = (((unsigned long long)P.sweep_hi << 32) | P.sweep_lo) + (unsigned long long)(gp / NB);
    t.sweep_lo = (uint32_t)sw; t.sweep_hi = (uint32_t)(sw >> 32);
    t.meas = MEAS && mode != 0 && pass >= w.passes - NB;   // the last sweep of the launch is the measured one
    t.y0 = ty * TY; t.ny = min(TY, L.Ly - t.y0);
    t.z0 = (int32_t)(((int64_t)zc * L.Lz) / w.n_zc); t.nz = (int32_t)(((int64_t)(zc + 1) * L.Lz) / w.n_zc) - t.z0;
    switch (b) {
      case 0: bw_tile<KIND, 0, V, TY, ROWB, kNB, ANISO, MEAS>(s, L, P, t, smem, sbase, rm, acc, n_acc, pending); break;
      case 1: bw_tile<KIND, 1, V, TY, ROWB, kNB, ANISO, MEAS>(s, L, P, t, smem, sbase, rm, acc, n_acc, pending); break;
      case 2: if constexpr (NB > 2) bw_tile<KIND, 2, V, TY, ROWB, kNB, ANISO, MEAS>(s, L, P, t, smem, sbase, rm, acc, n_acc, pending); break;
      default: if constexpr (NB > 3) bw_tile<KIND, 3, V, TY, ROWB, kNB, ANISO, MEAS>(s, L, P, t, smem, sbase, rm, acc, n_acc, pending); break;
    }
    if (pass + 1 < w.passes) {
      int32_t k = zc - pass % w.n_zc;   // position of the chunk in the pass's order (chunk = (k + pass) mod n)
      k = k < 0 ? k + w.n_zc : k;
      pending = w.done + (size_t)pass * w.n_zc + k;
    }
  }
}

template <int KIND, int V, int TY, int ROWB, int kNB, int MINB, int ANISO, bool MEAS>
__global__ void __launch_bounds__((bw_max_threads<V, TY, ROWB>()), MINB)
k_sweep_bravais_ws(float* s, BrLayout L, WsTiles w, SweepParams P, Meas m) {
  resolve_sweep(P);
  using S = BwSmem<KIND, TY, ROWB, kNB>;
  extern __shared__ __align__(128) unsigned char smem[];
  const uint32_t sbase = smem_u32(smem);
  const uint32_t n_cwarps = (blockDim.x >> 5) - 1;
  if (threadIdx.x == 0) {
    const uint32_t bar = sbase + S::OFF_BAR;
    for (int i = 0; i < kNB; ++i) { mbar_init(bar + 8u * i, 1); mbar_init(bar + 8u * (kNB + i), n_cwarps); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  double acc[4] = {0.0, 0.0, 0.0, 0.0};
  unsigned n_acc = 0;
  if (threadIdx.x < 32) bw_producer<KIND, TY, ROWB, kNB>(s, L, w, smem, sbase);
  else bw_consumer<KIND, V, TY, ROWB, kNB, ANISO, MEAS>(s, L, w, P, m.mode, smem, sbase, acc, n_acc);
  __shared__ uint32_t s_last;
  __syncthreads();
  if (threadIdx.x == 0) { __threadfence(); s_last = atomicAdd(w.sched + 1, 1u) == gridDim.x - 1 ? 1u : 0u; }
  __syncthreads();
  if (s_last) {   // the last CTA to finish re-arms the scheduler and clears the progress words
    __threadfence();
    for (int32_t i = threadIdx.x; i < (w.passes - 1) * w.n_zc; i += blockDim.x) w.done[i] = 0u;
    if (threadIdx.x == 0) { w.sched[0] = 0u; w.sched[1] = 0u; }
  }
  if (MEAS) {
    block_reduce4(acc[0], acc[1], acc[2], acc[3], m.partials + (size_t)blockIdx.x * 4);
    count_accepts(m.n_accept, n_acc);
  }
}

// ---- launch shapes ------------------------------------------------------------------------------------------------------
// rows of up to ROWB / 4 cells; V cells per thread; TY rows per tile; kNB groups in the ring; MINB CTAs per SM
//   bcc  Lx <=  64: V 2, 8 rows (256 consumer threads),  ring 4 x  6.9 KB, 3 CTAs/SM
//        Lx <= 128: V 4, 8 rows,                         ring 4 x 13.8 KB, 3 CTAs/SM
//        Lx <= 256: V 4, 4 rows,                         ring 4 x 15.4 KB, 3 CTAs/SM
//   fcc  Lx <=  64: V 2, 8 rows,                         ring 3 x 20.7 KB, 3 CTAs/SM
//        Lx <= 128: V 2, 4 rows (256 consumer threads),  ring 3 x 23.0 KB, 3 CTAs/SM   (c3)
//        Lx <= 256: V 4, 3 rows (192 consumer threads),  ring 3 x 36.9 KB, 2 CTAs/SM
struct BwShape { int V, TY, ROWB, kNB, MINB; };
__host__ constexpr BwShape bw_shape(int kind, int Lx) {
  if (kind == BR_BCC) return Lx <= 64 ? BwShape{4, 16, 256, 4, 3} : (Lx <= 128 ? BwShape{4, 8, 512, 4, 3} : BwShape{4, 4, 1024, 4, 3});
  return Lx <= 64 ? BwShape{4, 8, 256, 3, 3} : (Lx <= 128 ? BwShape{4, 4, 512, 3, 3} : BwShape{4, 3, 1024, 3, 2});
}

struct BwArgs { int passes, first, lag, n_zc, grid_cap; uint32_t* sched; uint32_t* done; };

template <int KIND, int V, int TY, int ROWB, int kNB, int MINB, int ANISO, bool MEAS>
cudaError_t bw_go(cudaStream_t st, float* s, const BrLayout& L, const SweepParams& p, const Meas& m, const BwArgs& a) {
  using S = BwSmem<KIND, TY, ROWB, kNB>;
  auto kern = k_sweep_bravais_ws<KIND, V, TY, ROWB, kNB, MINB, ANISO, MEAS>;
  static unsigned long long configured = 0;
  const cudaError_t e = ws_configure((const void*)kern, (int)S::BYTES, configured);
  if (e != cudaSuccess) return e;
  WsTiles w;
  w.n_ty = (L.Ly + TY - 1) / TY;
  w.n_zc = a.n_zc;
  w.sched = a.sched;
  w.passes = a.passes; w.lag = a.lag; w.first = a.first; w.done = a.done; w.zmask = 0xffffffffu;
  const long long n_tiles = (long long)w.n_ty * w.n_zc * a.passes;
  const long long cap = (long long)a.grid_cap * MINB;
  const int grid = (int)(n_tiles < cap ? n_tiles : cap);
  const int threads = 32 + 32 * ((TY * (L.Lx / V) + 31) / 32);
  return launch_colour_kernel(kern, dim3(grid), dim3(threads), S::BYTES, st, p.pdl != 0, s, L, w, p, m);
}

template <int KIND, int V, int TY, int ROWB, int kNB, int MINB>
cudaError_t bw_pick(cudaStream_t st, float* s, const BrLayout& L, const SweepParams& p, const Meas& m, const BwArgs& a) {
  if (m.mode != 0) return bw_go<KIND, V, TY, ROWB, kNB, MINB, ANISO_GENERAL, true>(st, s, L, p, m, a);   // general formula: the same bits
  const int aniso = (p.K == 0.0f) ? ANISO_NONE : ((p.ex == 0.0f && p.ey == 0.0f && p.ez == 1.0f) ? ANISO_Z : ANISO_GENERAL);
  switch (aniso) {
    case ANISO_NONE: return bw_go<KIND, V, TY, ROWB, kNB, MINB, ANISO_NONE, false>(st, s, L, p, m, a);
    case ANISO_Z: return bw_go<KIND, V, TY, ROWB, kNB, MINB, ANISO_Z, false>(st, s, L, p, m, a);
    default: return bw_go<KIND, V, TY, ROWB, kNB, MINB, ANISO_GENERAL, false>(st, s, L, p, m, a);
  }
}

}  // namespace

// rows of up to 256 cells, a multiple of 4 (16-byte bulk copies)
bool bravais_ws_supported(const BrLayout& L) { return !L.ghost && (L.kind == BR_BCC || L.kind == BR_FCC) && L.Lx % 4 == 0 && L.Lx <= 256; }

// chunks in z: ZT planes each (0: chosen so that one pass holds a few tiles per resident CTA)
int bravais_ws_chunks(const BrLayout& L, int ZT, int grid_cap) {
  if (ZT > 0) return (L.Lz + ZT - 1) / ZT;
  const BwShape sh = bw_shape(L.kind, L.Lx);
  const long long n_ty = (L.Ly + sh.TY - 1) / sh.TY, cap = (long long)grid_cap * sh.MINB;
  long long n = (4 * cap + n_ty - 1) / n_ty;             // about four tiles per CTA and pass
  if (n > L.Lz / 2) n = L.Lz / 2;                        // at least two planes per chunk (a group serves two steps)
  return (int)(n < 1 ? 1 : n);
}

// CTAs of a launch of `passes` colour passes (= block partials of its fused measurement)
int bravais_ws_blocks(const BrLayout& L, int ZT, int grid_cap, int passes) {
  const BwShape sh = bw_shape(L.kind, L.Lx);
  const long long n_tiles = (long long)((L.Ly + sh.TY - 1) / sh.TY) * bravais_ws_chunks(L, ZT, grid_cap) * passes;
  const long long cap = (long long)grid_cap * sh.MINB;
  return (int)(n_tiles < cap ? n_tiles : cap);
}

// `passes` colour passes starting with colour `first` of the sweep in p (first + passes may run over several sweeps);
// m.mode != 0: the last NB passes carry the fused measurement; done: kWsDoneWords device words, zero between launches
cudaError_t launch_sweep_bravais_ws(cudaStream_t st, float* s, BrLayout L, int ZT, int lag, int grid_cap, uint32_t* sched, uint32_t* done,
                                    SweepParams p, int first, int passes, Meas m) {
  if (!bravais_ws_supported(L) || passes < 1 || first < 0 || lag < 3) return cudaErrorInvalidValue;
  BwArgs a{passes, first, lag, bravais_ws_chunks(L, ZT, grid_cap), grid_cap, sched, done};
  if ((long long)(passes - 1) * a.n_zc > kWsDoneWords) return cudaErrorInvalidValue;
  if (L.kind == BR_BCC) {
    if (L.Lx <= 64) return bw_pick<BR_BCC, 4, 16, 256, 4, 3>(st, s, L, p, m, a);
    if (L.Lx <= 128) return bw_pick<BR_BCC, 4, 8, 512, 4, 3>(st, s, L, p, m, a);
    return bw_pick<BR_BCC, 4, 4, 1024, 4, 3>(st, s, L, p, m, a);
  }
  if (L.Lx <= 64) return bw_pick<BR_FCC, 4, 8, 256, 3, 3>(st, s, L, p, m, a);
  if (L.Lx <= 128) return bw_pick<BR_FCC, 4, 4, 512, 3, 3>(st, s, L, p, m, a);
  return bw_pick<BR_FCC, 4, 3, 1024, 3, 2>(st, s, L, p, m, a);
}

}  // namespace hb
