// hb_sc_ws.cu -- simple cubic colour pass, warp-specialised and persistent.
//
// Why: in the direct kernel (hb_kernels.cu) a third of the executed instructions are not the update at
// all but the memory side of it -- 64-bit address arithmetic for 24 global accesses and 12 prefetches per
// thread and plane -- and the board runs at its power cap, so instructions are what the sustained rate pays
// for.  Here the memory side is moved out of the update warps:
//
//   * one PRODUCER warp per CTA streams whole lattice rows into shared memory with 1-D bulk asynchronous
//     copies (cp.async.bulk, the TMA engine), completing on mbarriers: a ring of NB plane slots of the
//     other colour (rows y0-1 .. y0+TY);
//   * the CONSUMER warps wait on a "full" barrier, read everything with LDS at compile-time offsets (row
//     pitch ROWB is a template constant, the periodic wrap in x is an index inside the staged row), release
//     the slots through "empty" barriers, run the attempt arithmetic of hb_device.cuh; their own spins they
//     load themselves (LDG.128; one plane ahead in the variants that have the registers for it) and store
//     with STG.128 at the same addresses.  No block-wide barrier in the steady state;
//   * CTAs are persistent (one to three per SM): a CTA takes tiles (TY rows x a chunk of planes) from a device counter,
//     one after the other, with the rings running across tile boundaries, so the pipeline is filled once per launch,
//     not once per tile, and no CTA is left with a fixed share when its SM runs slower than the others.
//
// Same arithmetic, same order of the neighbour sum, same bits as k_sweep_sc.
//
// FUSED (sc_kernel = 2): ONE launch runs several colour passes -- both colours of a sweep, or of several
// sweeps -- as one stream of tiles with dependencies between them instead of a launch boundary after every colour
// (the multi-colour tile kernel; the on-chip memory that carries the freshly written colour from one
// pass to the next is the 126 MB L2 rather than shared memory, so no halo is recomputed and the update stays in place).
// Pass p = (sweep p/2, colour p%2) walks the z-chunks in the order p, p+1, ... (mod n: the rotation makes the
// periodic wrap in z a dependency on an EARLIER chunk), `lag` rounds behind pass p-1; its k-th chunk may start when pass
// p-1 has finished its chunks k, k+1, k+2 (the planes it reads as neighbours, and the readers of what it overwrites).
// Tiles are handed out in round order from the same device counter, so every dependency of a tile was handed out
// before it: the oldest unfinished tile can always run, whatever the CTAs hold.
#include "hb_device.cuh"
#include "hb_internal.h"
#include "hb_ws.cuh"

// HB_WS_HOIST: how many of the four Philox draws of a plane step a consumer makes before it waits for the staged planes
// (0, 2 or 4, "interleave").  Measured in round 3; the default is what won.
#ifndef HB_WS_HOIST
#define HB_WS_HOIST 0
#endif

namespace hb {

namespace {


// threads of a CTA the kernel is compiled for: the producer warp plus TY rows of ROWB/16 vectors; the 7-row shape is built
// for rows of at most 59 vectors (13 consumer warps: 448 threads, two CTAs per SM at 72 registers)
template <int TY, int ROWB>
__host__ __device__ constexpr int ws_max_threads() {
  if (TY == 7) return 32 + 32 * 13;
  const int t = 32 + 32 * ((TY * (ROWB / 16) + 31) / 32);
  return t > 1024 ? 1024 : t;
}
// own spins one plane ahead in registers: only where the register budget allows (4-row tiles, 2 CTAs per SM)
template <int TY, int MINB>
__host__ __device__ constexpr bool ws_pref() { return MINB < 3 && TY != 7; }

// slab with neighbour flags: the two boundary chunks (the first and the last in z) are handed out first
__device__ __forceinline__ int32_t ws_chunk_in_order(int32_t q, int32_t n_zc, bool boundary_first) {
  if (!boundary_first || n_zc < 3) return q;
  return q == 0 ? 0 : (q == 1 ? n_zc - 1 : q - 1);
}
__device__ __forceinline__ uint32_t ld_acquire_sys(const uint32_t* p) {
  uint32_t v;
  asm volatile("ld.acquire.sys.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_release_sys(uint32_t* p, uint32_t v) {
  asm volatile("st.release.sys.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

// kNB plane slots of the other colour (z-1, z, z+1 and look-ahead); MINB = CTAs per SM the kernel is built for
template <int TY, int ROWB, int kNB, int MINB>
struct WsSmem {
  static constexpr uint32_t SLOT_B = 3u * (TY + 2) * ROWB;
  static constexpr uint32_t OFF_BAR = kNB * SLOT_B;   // full[kNB], empty[kNB]
  static constexpr uint32_t OFF_TILE = OFF_BAR + 8u * (2 * kNB);   // info[kNB]: the tile a staged plane belongs to (x = tile, -1 = no more
                                                                    // tiles; fused launches: y = pass, z = chunk, w = tile in y)
  static constexpr uint32_t BYTES = OFF_TILE + 16u * kNB;
  static_assert((OFF_TILE % 16u) == 0, "tile info alignment");
};

// ---- producer: one warp ------------------------------------------------------------------------------
// plane k of a tile is lattice plane z0-1+k (periodic), rows y0-1 .. y0+ny (periodic) of the other colour
template <int TY, int ROWB, int kNB, int MINB, bool FUSED, bool ALIAS>
__device__ __forceinline__ void ws_producer(const float* b, const ScLayout& L, const WsTiles& w,
                                            unsigned char* smem, uint32_t sbase) {
  using S = WsSmem<TY, ROWB, kNB, MINB>;
  const uint32_t lane = threadIdx.x;
  const uint32_t row_bytes = (uint32_t)L.H * 4u;
  const size_t n = L.n;
  const uint32_t fullB = sbase + S::OFF_BAR, emptyB = fullB + 8u * kNB;
  RingPos<kNB> rp;   // next plane slot to fill
  const int32_t n_tiles = w.n_ty * w.n_zc * (FUSED ? w.passes : 1);
  volatile int4* info = reinterpret_cast<volatile int4*>(smem + S::OFF_TILE);
  const float* const spins = b;   // FUSED: b is the base of the spins; the colour a tile reads depends on its pass
  // Tiles are handed out dynamically (one atomic per tile): the CTAs of a launch do not run at the same speed, and with a
  // fixed share per CTA the fast SMs idled at the end of every launch (ncu: SMs active 70-99 % of the launch).  The
  // consumers learn the tile from a word written beside the plane slot before the slot's "full" barrier is armed.
  for (;;) {
    int32_t tile = 0;
    if (lane == 0) tile = (int32_t)atomicAdd(w.sched, 1u);
    tile = __shfl_sync(0xffffffffu, tile, 0);
    if (tile >= n_tiles) {   // tell the consumers: the slot they will wait on next carries no plane
      mbar_wait_backoff(emptyB + 8u * rp.slot, rp.par ^ 1u);
      if (lane == 0) { info[rp.slot].x = -1; mbar_arrive(fullB + 8u * rp.slot); }
      break;
    }
    int32_t ty = tile % w.n_ty, zc = ws_chunk_in_order(tile / w.n_ty, w.n_zc, L.flag_in != nullptr), pass = 0;
    if (!FUSED && L.flag_in) {   // a boundary tile of a slab: the neighbour on that side must be through its boundary chunk of the pass before
      const bool lo = zc == 0, hi = zc == w.n_zc - 1;
      if (lo || hi) {
        if (lane == 0 && lo) while ((int32_t)(ld_acquire_sys(L.flag_in) - (L.stamp - 1u)) < 0) __nanosleep(200);
        if (lane == 1 && hi) while ((int32_t)(ld_acquire_sys(L.flag_in + 1) - (L.stamp - 1u)) < 0) __nanosleep(200);
        __syncwarp();
        asm volatile("fence.proxy.async;" ::: "memory");   // the bulk copies below read the ghost plane the neighbour stored
      }
    }
    if (FUSED) {
      const FusedTile t = fused_decode(tile, w);
      ty = t.ty; zc = t.zc; pass = t.p;
      if (t.p > 0) {   // the chunks of the previous pass this tile reads, and whose readers must be done before it writes
        if (lane < 3) {
          const uint32_t* d = w.done + (size_t)(t.p - 1) * w.n_zc + (t.k + (int32_t)lane) % w.n_zc;
          const uint32_t all = (uint32_t)w.n_ty * ((blockDim.x >> 5) - 1u);
          while (ld_acquire_gpu(d) < all) __nanosleep(256);
        }
        __syncwarp();
        asm volatile("fence.proxy.async;" ::: "memory");   // the bulk copies below read what other CTAs stored (generic proxy)
      }
      b = spins + (size_t)(1 - (t.p & 1)) * L.half;          // pass p updates colour p % 2 and reads the other one
    }
    const int32_t y0 = ty * TY, ny = min(TY, L.Ly - y0);
    const int32_t z0 = (int32_t)(((int64_t)zc * L.Lz) / w.n_zc), nz = (int32_t)(((int64_t)(zc + 1) * L.Lz) / w.n_zc) - z0;
    for (int32_t k = 0; k < nz + 2; ++k) {
      {  // B plane k
        int32_t zz = z0 - 1 + k;
        zz = zz < 0 ? zz + L.Lz : (zz >= L.Lz ? zz - L.Lz : zz);
        const uint32_t slot = rp.slot;
        mbar_wait_backoff(emptyB + 8u * slot, rp.par ^ 1u);
        const uint32_t n_rows = 3u * (uint32_t)(ny + 2);
        if (lane == 0) {
          info[slot].x = tile; info[slot].y = pass; info[slot].z = zc; info[slot].w = ty;
          mbar_expect_tx(fullB + 8u * slot, n_rows * row_bytes);
        }
        __syncwarp();
        for (uint32_t q = lane; q < n_rows; q += 32) {
          const uint32_t comp = q / (uint32_t)(ny + 2), r = q - comp * (uint32_t)(ny + 2);
          int32_t yy = y0 - 1 + (int32_t)r;
          yy = yy < 0 ? yy + L.Ly : (yy >= L.Ly ? yy - L.Ly : yy);
          const float* src = b + comp * n + ((size_t)(ALIAS ? (int32_t)((uint32_t)zz & w.zmask) : zz) * L.Ly + yy) * L.H;
          bulk_g2s(sbase + slot * S::SLOT_B + (comp * (TY + 2) + r) * ROWB, src, row_bytes, fullB + 8u * slot);
        }
        rp.next();
      }
    }
  }
}

// ---- consumers -------------------------------------------------------------------------------------------
template <int TY, int ROWB, int kNB, int MINB, int ANISO, bool MEAS, bool SLAB, bool FUSED, bool ALIAS>
__device__ __forceinline__ void ws_consumer(float* a, const ScLayout& L, const WsTiles& w, const SweepParams& P, int colour,
                                            int mode, unsigned char* smem, uint32_t sbase, double acc[4], unsigned& n_acc) {
  using S = WsSmem<TY, ROWB, kNB, MINB>;
  const uint32_t fullB = sbase + S::OFF_BAR, emptyB = fullB + 8u * kNB;
  const int32_t HV = L.H >> 2;
  const int32_t c = (int32_t)threadIdx.x - 32;
  const int32_t r = c / HV, j = c - r * HV;
  const int32_t i0 = j * 4;
  const bool lane0 = (threadIdx.x & 31) == 0;
  // byte offsets inside a plane slot (component 0): the thread's row is row r+1 of the slot
  const uint32_t t_row = (uint32_t)(r + 1) * ROWB;
  const uint32_t t_off = t_row + (uint32_t)j * 16u;
  const uint32_t h_lo = t_row + (uint32_t)(i0 == 0 ? L.H - 1 : i0 - 1) * 4u;        // p = 0: element i0-1 (periodic)
  const uint32_t h_hi = t_row + (uint32_t)(i0 + 4 >= L.H ? i0 + 4 - L.H : i0 + 4) * 4u;  // p = 1: element i0+4
  const size_t n = L.n;
  const size_t plane = (size_t)L.Ly * L.H;
  RingPos<kNB> rm;   // slot of plane z-1 of the current step; rc, rq (planes z, z+1) are carried beside it: one next() per step
  RingPos<kNB> rc = rm; rc.next();
  RingPos<kNB> rq = rc; rq.next();
  const volatile int4* info = reinterpret_cast<const volatile int4*>(smem + S::OFF_TILE);
  float* const spins = a;   // FUSED: a is the base of the spins; the colour a tile updates depends on its pass
  uint32_t sweep_lo = P.sweep_lo, sweep_hi = P.sweep_hi;
  int32_t pass = 0;
  // FUSED: the progress word this warp still has to bump for the tile it finished last.  The bump needs a device-wide
  // fence behind the tile's stores; issued right after them the fence waits ~1 us for their acknowledgement (ncu: 7 % of
  // the warps' time in membar).  So it is deferred to just before the first stores of the NEXT tile, one plane of
  // arithmetic later, when the earlier stores have long been acknowledged.
  uint32_t* pending = nullptr;
  auto publish = [&]() {
    __syncwarp();
    if (lane0) {
      asm volatile("fence.proxy.async;" ::: "memory");   // the waiting CTAs read these stores with bulk copies (async proxy)
      __threadfence();
      atomicAdd(pending, 1u);
    }
    pending = nullptr;
  };
  for (;;) {
    if (FUSED && pending) {
      // Deferring is only safe once the producer is past the dependencies of the next tile (they may include the very
      // tile this warp has not published yet): that is the case when the tile's first plane has been staged.
      uint32_t staged = 0;
      if (lane0) staged = mbar_test(fullB + 8u * rm.slot, rm.par) ? 1u : 0u;
      if (!__shfl_sync(0xffffffffu, staged, 0)) publish();
    }
    mbar_wait(fullB + 8u * rm.slot, rm.par);   // first plane of the next tile, or the producer's "no more tiles"
    const int32_t tile = info[rm.slot].x;
    if (tile < 0) { if (FUSED && pending) publish(); break; }
    int32_t ty = tile % w.n_ty, zc = ws_chunk_in_order(tile / w.n_ty, w.n_zc, SLAB && L.flag_in != nullptr);
    if (FUSED) {
      pass = info[rm.slot].y; zc = info[rm.slot].z; ty = info[rm.slot].w;
      colour = pass & 1;
      a = spins + (size_t)colour * L.half;
      const unsigned long long sw = (((unsigned long long)P.sweep_hi << 32) | P.sweep_lo) + (unsigned long long)(pass >> 1);
      sweep_lo = (uint32_t)sw; sweep_hi = (uint32_t)(sw >> 32);
      if (MEAS) mode = pass == w.passes - 1 ? 2 : (pass == w.passes - 2 ? 1 : 0);   // the last sweep of the launch is the measured one
    }
    const int32_t y0 = ty * TY, ny = min(TY, L.Ly - y0);
    const int32_t z0 = (int32_t)(((int64_t)zc * L.Lz) / w.n_zc), nz = (int32_t)(((int64_t)(zc + 1) * L.Lz) / w.n_zc) - z0;
    const bool active = r < ny;
    const int32_t y = y0 + r;
    float* gx = a + ((size_t)(ALIAS ? (int32_t)((uint32_t)z0 & w.zmask) : z0) * L.Ly + y) * L.H + i0;   // own spins of plane z0 (x component)
    uint32_t site_row = (uint32_t)(z0 * L.Ly + y) * (uint32_t)L.Lx + 2u * (uint32_t)i0 + L.site_base;
    // own spins come straight from global memory, one plane ahead of their use (only this thread writes them)
    constexpr bool PREF = ws_pref<TY, MINB>();   // otherwise (72 registers) the other warps cover the latency instead
    Vec<4> nxt[3];
    if (PREF && active) { nxt[0] = load_rw<4>(gx); nxt[1] = load_rw<4>(gx + n); nxt[2] = load_rw<4>(gx + 2 * n); }
    for (int32_t s = 0; s < nz; ++s) {
      // ghost planes of a slab are staged as neighbours but not updated: the z-neighbour owns them
      const int32_t zs = z0 + s;
      const bool act = active && !(SLAB && (zs == 0 || zs == L.Lz - 1));
      Vec<4> sp[3];
      if (PREF) {
        sp[0] = nxt[0]; sp[1] = nxt[1]; sp[2] = nxt[2];
        if (active && s + 1 < nz) {
          nxt[0] = load_rw<4>(gx + plane); nxt[1] = load_rw<4>(gx + plane + n); nxt[2] = load_rw<4>(gx + plane + 2 * n);
        }
      } else if (act) {
        if (FUSED) {   // an earlier pass of this launch, on any SM, wrote them: read at the L2, never a line kept in this SM's L1
          sp[0] = load_cg<4>(gx); sp[1] = load_cg<4>(gx + n); sp[2] = load_cg<4>(gx + 2 * n);
        } else {
          sp[0] = load_rw<4>(gx); sp[1] = load_rw<4>(gx + n); sp[2] = load_rw<4>(gx + 2 * n);
        }
      }
      const int32_t p = (colour + y + z0 + s) & 1;
#if HB_WS_HOIST > 0
      // the random words of the first HB_WS_HOIST attempts of this plane step, drawn BEFORE the wait for the staged planes: the
      // IMAD.WIDE bursts of Philox then run while other warps are in their LDS phase instead of colliding with theirs
      Rand4 pre[HB_WS_HOIST];
      if (act) {
#pragma unroll
        for (int j = 0; j < HB_WS_HOIST; ++j)
          pre[j] = philox4x32_10(site_row + (uint32_t)p + 2u * j, 0u, sweep_lo, sweep_hi, P.seed_lo, P.seed_hi);
      }
#endif
      if (s == 0) mbar_wait(fullB + 8u * rc.slot, rc.par);
      mbar_wait(fullB + 8u * rq.slot, rq.par);
      const unsigned char* Bm = smem + rm.slot * S::SLOT_B;
      const unsigned char* Bc = smem + rc.slot * S::SLOT_B;
      const unsigned char* Bp = smem + rq.slot * S::SLOT_B;
      const uint32_t h_off = p ? h_hi : h_lo;
      Vec<4> h[3];
      if (act) {
#pragma unroll
        for (int q = 0; q < 3; ++q) {
          constexpr uint32_t CB = (TY + 2) * ROWB;
          const float4 cc = *reinterpret_cast<const float4*>(Bc + q * CB + t_off);
          const float halo = *reinterpret_cast<const float*>(Bc + q * CB + h_off);
          const float4 ym = *reinterpret_cast<const float4*>(Bc + q * CB + t_off - ROWB);
          const float4 yp = *reinterpret_cast<const float4*>(Bc + q * CB + t_off + ROWB);
          const float4 zm = *reinterpret_cast<const float4*>(Bm + q * CB + t_off);
          const float4 zp = *reinterpret_cast<const float4*>(Bp + q * CB + t_off);
          // -x,+x,-y,+y,-z,+z: the two x terms are elements i-1+p and i+p of the row (they commute bitwise)
          const f2 sel_lo = make_float2(p ? cc.y : halo, p ? cc.z : cc.x);
          const f2 sel_hi = make_float2(p ? cc.w : cc.y, p ? halo : cc.z);
          f2 u = add2(make_float2(cc.x, cc.y), sel_lo), v = add2(make_float2(cc.z, cc.w), sel_hi);
          u = add2(u, make_float2(ym.x, ym.y)); v = add2(v, make_float2(ym.z, ym.w));
          u = add2(u, make_float2(yp.x, yp.y)); v = add2(v, make_float2(yp.z, yp.w));
          u = add2(u, make_float2(zm.x, zm.y)); v = add2(v, make_float2(zm.z, zm.w));
          u = add2(u, make_float2(zp.x, zp.y)); v = add2(v, make_float2(zp.z, zp.w));
          h[q] = Vec<4>{{u.x, u.y, v.x, v.y}};
        }
      }
      // this warp is done with plane z-1 (after the last plane of a tile: with all three)
      __syncwarp();
      if (lane0) {
        mbar_arrive(emptyB + 8u * rm.slot);
        if (s == nz - 1) {
          mbar_arrive(emptyB + 8u * rc.slot);
          mbar_arrive(emptyB + 8u * rq.slot);
        }
      }
      bool any_acc = false;
      if (act) {
        const uint32_t site0 = site_row + (uint32_t)p;
#pragma unroll
        for (int k = 0; k < 4; k += 2) {
#if HB_WS_HOIST > 0
          const Rand4 ra = k < HB_WS_HOIST ? pre[k < HB_WS_HOIST ? k : 0] : philox4x32_10(site0 + 2u * k, 0u, sweep_lo, sweep_hi, P.seed_lo, P.seed_hi);
          const Rand4 rb = k + 1 < HB_WS_HOIST ? pre[k + 1 < HB_WS_HOIST ? k + 1 : 0] : philox4x32_10(site0 + 2u * k + 2u, 0u, sweep_lo, sweep_hi, P.seed_lo, P.seed_hi);
#else
          const Rand4 ra = philox4x32_10(site0 + 2u * k, 0u, sweep_lo, sweep_hi, P.seed_lo, P.seed_hi);
          const Rand4 rb = philox4x32_10(site0 + 2u * k + 2u, 0u, sweep_lo, sweep_hi, P.seed_lo, P.seed_hi);
#endif
          f2 px = make_float2(sp[0].v[k], sp[0].v[k + 1]), py = make_float2(sp[1].v[k], sp[1].v[k + 1]),
             pz = make_float2(sp[2].v[k], sp[2].v[k + 1]);
          bool acc_a, acc_b;
          attempt2<ANISO>(ra, rb, P.J, P.K, P.beta, P.ex, P.ey, P.ez, make_float2(h[0].v[k], h[0].v[k + 1]),
                          make_float2(h[1].v[k], h[1].v[k + 1]), make_float2(h[2].v[k], h[2].v[k + 1]), px, py, pz, acc_a, acc_b);
          sp[0].v[k] = px.x; sp[0].v[k + 1] = px.y; sp[1].v[k] = py.x; sp[1].v[k + 1] = py.y;
          sp[2].v[k] = pz.x; sp[2].v[k + 1] = pz.y;
          any_acc |= acc_a | acc_b;
          if (MEAS && (!FUSED || mode != 0)) n_acc += (unsigned)acc_a + (unsigned)acc_b;
        }
      }
      if (FUSED && pending) publish();   // (outside the divergent part: the whole warp)
      if (act) {
        if (any_acc) {
          store<4>(gx, sp[0]);
          store<4>(gx + n, sp[1]);
          store<4>(gx + 2 * n, sp[2]);
          if (SLAB) {   // slab with peer stores: the boundary planes go straight into the neighbours' ghost planes
            const bool lo = zs == 1, hi = zs == L.Lz - 2;
            float* pb = lo ? L.peer[0] : (hi ? L.peer[1] : nullptr);
            if (pb) {
              const uint32_t pn = lo ? L.peer_n[0] : L.peer_n[1], ph = lo ? L.peer_half[0] : L.peer_half[1];
              float* q = pb + (size_t)colour * ph + (lo ? L.peer_zoff[0] : L.peer_zoff[1]) + (size_t)y * L.H + i0;
              store<4>(q, sp[0]);
              store<4>(q + pn, sp[1]);
              store<4>(q + 2 * (size_t)pn, sp[2]);
            }
          }
        }
        if (MEAS && (!FUSED || mode != 0)) {
          float mx = 0.0f, my = 0.0f, mz = 0.0f, me = 0.0f;
          const float Jx = (mode == 2) ? -P.J : 0.0f;
#pragma unroll
          for (int k = 0; k < 4; ++k) {
            mx = __fadd_rn(mx, sp[0].v[k]); my = __fadd_rn(my, sp[1].v[k]); mz = __fadd_rn(mz, sp[2].v[k]);
            const float sh = __fmaf_rn(sp[2].v[k], h[2].v[k], __fmaf_rn(sp[1].v[k], h[1].v[k], __fmul_rn(sp[0].v[k], h[0].v[k])));
            const float e = __fmaf_rn(sp[2].v[k], P.ez, __fmaf_rn(sp[1].v[k], P.ey, __fmul_rn(sp[0].v[k], P.ex)));
            me = __fadd_rn(me, __fmaf_rn(Jx, sh, __fmul_rn(-P.K, __fmul_rn(e, e))));
          }
          acc[0] += (double)mx; acc[1] += (double)my; acc[2] += (double)mz; acc[3] += (double)me;
        }
      }
      if (ALIAS) gx = a + ((size_t)((uint32_t)(z0 + s + 1) & w.zmask) * L.Ly + y) * L.H + i0; else gx += plane;
      site_row += (uint32_t)(L.Ly * L.Lx);
      rm = rc; rc = rq; rq.next();
    }
    rm = rq; rc = rm; rc.next(); rq = rc; rq.next();   // past the two extra planes of the tile
    if (SLAB && L.flag_in) {
      // a boundary tile is done: the last warp of the last tile of a boundary chunk tells the neighbour on that side
      const bool lo = zc == 0, hi = zc == w.n_zc - 1;
      if (lo || hi) {
        __syncwarp();
        if (lane0) {
          __threadfence_system();   // this warp's stores, the ones into the neighbour's ghost plane included
          const uint32_t all = (uint32_t)w.n_ty * ((blockDim.x >> 5) - 1u);
#pragma unroll
          for (int side = 0; side < 2; ++side)
            if (side == 0 ? lo : hi)
              if (atomicAdd(L.bnd_count + side, 1u) == all - 1u) {
                L.bnd_count[side] = 0u;
                __threadfence_system();
                st_release_sys(L.flag_out[side], L.stamp);
              }
        }
      }
    }
    if (FUSED && pass + 1 < w.passes) {
      // this warp's stores of the tile are done: the next pass waits for the chunk's progress word (see publish above)
      int32_t k = zc - pass % w.n_zc;   // position of the chunk in the pass's order (chunk = (k + pass) mod n)
      k = k < 0 ? k + w.n_zc : k;
      pending = w.done + (size_t)pass * w.n_zc + k;
    }
  }
}

// SLAB: the lattice is a slab of a larger one (ScLayout::ghost): its first and last planes are ghost planes, staged as
// neighbours but not updated, and boundary-plane stores are repeated into the z-neighbours' buffers (hb_slab_set_peer).
// A separate instantiation: the whole-lattice kernel carries none of it.
template <int TY, int ROWB, int kNB, int MINB, int ANISO, bool MEAS, bool SLAB, bool FUSED, bool ALIAS>
__global__ void __launch_bounds__((ws_max_threads<TY, ROWB>()), MINB)
k_sweep_sc_ws(float* a, const float* b, ScLayout L, WsTiles w, SweepParams P, int colour, Meas m) {
  resolve_sweep(P);
  using S = WsSmem<TY, ROWB, kNB, MINB>;
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
  if (threadIdx.x < 32) ws_producer<TY, ROWB, kNB, MINB, FUSED, ALIAS>(b, L, w, smem, sbase);
  else ws_consumer<TY, ROWB, kNB, MINB, ANISO, MEAS, SLAB, FUSED, ALIAS>(a, L, w, P, colour, m.mode, smem, sbase, acc, n_acc);
  if (FUSED) {
    // the last CTA to finish re-arms the scheduler and clears the progress words; all of its warps must be through first
    __shared__ uint32_t s_last;
    __syncthreads();
    if (threadIdx.x == 0) { __threadfence(); s_last = atomicAdd(w.sched + 1, 1u) == gridDim.x - 1 ? 1u : 0u; }
    __syncthreads();
    if (s_last) {
      __threadfence();
      for (int32_t i = threadIdx.x; i < w.passes * w.n_zc; i += blockDim.x) w.done[i] = 0u;
      if (threadIdx.x == 0) { w.sched[0] = 0u; w.sched[1] = 0u; }
    }
  } else if (threadIdx.x == 0) {   // this thread took the CTA's last tile number above; the last CTA to finish re-arms the scheduler
    __threadfence();
    if (atomicAdd(w.sched + 1, 1u) == gridDim.x - 1) { w.sched[0] = 0u; w.sched[1] = 0u; }
  }
  if (MEAS) {
    block_reduce4(acc[0], acc[1], acc[2], acc[3], m.partials + (size_t)blockIdx.x * 4);
    count_accepts(m.n_accept, n_acc);
  }
}

struct FusedArgs { int passes, lag; uint32_t* done; uint32_t zmask = 0xffffffffu; };   // passes = 0: a plain launch of one colour

template <int TY, int ROWB, int kNB, int MINB, int ANISO, bool MEAS, bool SLAB = false, bool FUSED = false, bool ALIAS = false>
cudaError_t ws_go(cudaStream_t st, float* s, const ScLayout& L, int n_zc, int grid_cap, uint32_t* sched, const SweepParams& p, int colour, const Meas& m,
                  const FusedArgs& f = FusedArgs{0, 0, nullptr}) {
  using S = WsSmem<TY, ROWB, kNB, MINB>;
  auto kern = k_sweep_sc_ws<TY, ROWB, kNB, MINB, ANISO, MEAS, SLAB, FUSED, ALIAS>;
  static unsigned long long configured = 0;
  const cudaError_t e = ws_configure((const void*)kern, (int)S::BYTES, configured);
  if (e != cudaSuccess) return e;
  WsTiles w;
  w.n_ty = (L.Ly + TY - 1) / TY;
  w.n_zc = n_zc;
  w.sched = sched;
  w.passes = f.passes; w.lag = f.lag; w.done = f.done; w.zmask = f.zmask; w.first = 0;
  const long long n_tiles = (long long)w.n_ty * w.n_zc * (FUSED ? f.passes : 1);
  const int grid = n_tiles < grid_cap ? (int)n_tiles : grid_cap;
  const int threads = 32 + 32 * ((TY * (L.H / 4) + 31) / 32);
  if (FUSED)   // the kernel picks the colour planes per tile from the base of the spins
    return launch_colour_kernel(kern, dim3(grid), dim3(threads), S::BYTES, st, p.pdl != 0, s, s, L, w, p, 0, m);
  float* a = s + (size_t)colour * L.half;
  const float* b = s + (size_t)(1 - colour) * L.half;
  return launch_colour_kernel(kern, dim3(grid), dim3(threads), S::BYTES, st, p.pdl != 0, a, b, L, w, p, colour, m);
}

template <int TY, int ROWB, int kNB, int MINB>
cudaError_t ws_pick(cudaStream_t st, float* s, const ScLayout& L, int n_zc, int grid_cap, uint32_t* sched, const SweepParams& p, int colour, const Meas& m,
                    const FusedArgs& f = FusedArgs{0, 0, nullptr}) {
  const int aniso = (p.K == 0.0f) ? ANISO_NONE : ((p.ex == 0.0f && p.ey == 0.0f && p.ez == 1.0f) ? ANISO_Z : ANISO_GENERAL);
  if (f.passes > 0) {   // several colour passes in one launch (whole lattices only)
    if (L.ghost) return cudaErrorInvalidValue;
    if (m.mode != 0) {
      switch (aniso) {
        case ANISO_NONE: return ws_go<TY, ROWB, kNB, MINB, ANISO_NONE, true, false, true>(st, s, L, n_zc, grid_cap, sched, p, colour, m, f);
        case ANISO_Z: return ws_go<TY, ROWB, kNB, MINB, ANISO_Z, true, false, true>(st, s, L, n_zc, grid_cap, sched, p, colour, m, f);
        default: return ws_go<TY, ROWB, kNB, MINB, ANISO_GENERAL, true, false, true>(st, s, L, n_zc, grid_cap, sched, p, colour, m, f);
      }
    }
    switch (aniso) {
      case ANISO_NONE: return ws_go<TY, ROWB, kNB, MINB, ANISO_NONE, false, false, true>(st, s, L, n_zc, grid_cap, sched, p, colour, m, f);
      case ANISO_Z: return ws_go<TY, ROWB, kNB, MINB, ANISO_Z, false, false, true>(st, s, L, n_zc, grid_cap, sched, p, colour, m, f);
      default: return ws_go<TY, ROWB, kNB, MINB, ANISO_GENERAL, false, false, true>(st, s, L, n_zc, grid_cap, sched, p, colour, m, f);
    }
  }
  if (L.ghost) {   // slab contexts measure with the separate pass
    if (m.mode != 0) return cudaErrorInvalidValue;
    switch (aniso) {
      case ANISO_NONE: return ws_go<TY, ROWB, kNB, MINB, ANISO_NONE, false, true>(st, s, L, n_zc, grid_cap, sched, p, colour, m);
      case ANISO_Z: return ws_go<TY, ROWB, kNB, MINB, ANISO_Z, false, true>(st, s, L, n_zc, grid_cap, sched, p, colour, m);
      default: return ws_go<TY, ROWB, kNB, MINB, ANISO_GENERAL, false, true>(st, s, L, n_zc, grid_cap, sched, p, colour, m);
    }
  }
  if (m.mode != 0) {
    switch (aniso) {
      case ANISO_NONE: return ws_go<TY, ROWB, kNB, MINB, ANISO_NONE, true>(st, s, L, n_zc, grid_cap, sched, p, colour, m);
      case ANISO_Z: return ws_go<TY, ROWB, kNB, MINB, ANISO_Z, true>(st, s, L, n_zc, grid_cap, sched, p, colour, m);
      default: return ws_go<TY, ROWB, kNB, MINB, ANISO_GENERAL, true>(st, s, L, n_zc, grid_cap, sched, p, colour, m);
    }
  }
  switch (aniso) {
    case ANISO_NONE: return ws_go<TY, ROWB, kNB, MINB, ANISO_NONE, false>(st, s, L, n_zc, grid_cap, sched, p, colour, m);
    case ANISO_Z: return ws_go<TY, ROWB, kNB, MINB, ANISO_Z, false>(st, s, L, n_zc, grid_cap, sched, p, colour, m);
    default: return ws_go<TY, ROWB, kNB, MINB, ANISO_GENERAL, false>(st, s, L, n_zc, grid_cap, sched, p, colour, m);
  }
}

}  // namespace

// rows of up to 256 floats per colour (Lx <= 512), a multiple of 4: the staged row pitch is 1024 bytes
bool sc_ws_supported(const ScLayout& L) { return L.H % 4 == 0 && L.H <= 256; }

// variants (option sc_ws_variant), sustained rate on c4 (sc L = 464) beside the direct kernel's 116.8 Gupd/s:
//   2 = 4-row tiles, 4 plane slots, 3 CTAs per SM, 72 registers, own spins loaded at the top of the step   120.9
//   0 = 4-row tiles, 5 plane slots, 2 CTAs per SM, 96 registers, own spins loaded one plane ahead          116.9
//   1 = 8-row tiles, 6 plane slots, 1 CTA per SM                                                            117.4
//   3 = 16-row tiles, 4 plane slots (216 KB), 1 CTA per SM of up to 31 consumer warps, 64 registers: for rows of up to
//       248 floats; with 232-float rows (c4) the 928 consumer threads are exactly 29 full warps
// (11-row tiles, whose 638 consumer threads fill 99.7 % of their warps' lanes, 1 CTA per SM: 111-113)
//   4 = 7-row tiles, 4 plane slots (108 KB), 2 CTAs per SM of 13 consumer warps, 72 registers: for rows of up to 236
//       floats; with 232-float rows (c4) 406 of the 416 consumer lanes work (97.6 %, against 90.6 % of the 4-row tile)
//   5 = 8-row tiles at a row pitch of 512 bytes, 4 plane slots (61 KB), 3 CTAs per SM of 8 consumer warps: for rows of up to
//       128 floats (Lx <= 256); with 128-float rows every consumer lane works
static int ws_ty(int variant) { return (variant == 1 || variant == 5) ? 8 : (variant == 3 ? 16 : (variant == 4 ? 7 : 4)); }
static int ws_ctas_per_sm(int variant) { return (variant == 1 || variant == 3) ? 1 : ((variant == 2 || variant == 5) ? 3 : 2); }

bool sc_ws_variant_supported(const ScLayout& L, int variant) {
  if (variant < 0 || variant > 5 || !sc_ws_supported(L)) return false;
  if (variant == 5) return L.H <= 128;              // row pitch of 512 bytes
  if (variant == 3) return 16 * (L.H / 4) <= 992;   // 1024 threads less the producer warp
  if (variant == 4) return 7 * (L.H / 4) <= 416;    // 13 consumer warps
  return true;
}

// Chunks in z of one launch.  ZT > 0: chunks of at most ZT planes.  ZT = 0: the count that minimises the longest
// walk of a CTA, rounds x (planes per chunk + 2): the persistent CTAs take the tiles in order, a tile costs its planes
// plus the two extra planes the producer stages for it (measured on c4, 7-row tiles: 13 chunks 130.7 Gupd/s, chunks of
// 24 / 16 / 12 / 8 planes 128.7 / 127 / 128 / 128).
int sc_ws_chunks(const ScLayout& L, int ZT, int grid_cap, int variant) {
  if (ZT > 0) return (L.Lz + ZT - 1) / ZT;
  const int ty = ws_ty(variant);
  const long long n_ty = (L.Ly + ty - 1) / ty, cap = (long long)grid_cap * ws_ctas_per_sm(variant);
  long long best = -1; int best_n = 1;
  const int n_max = L.Lz < 4096 ? L.Lz : 4096;
  for (int n = 1; n <= n_max; ++n) {
    const long long tiles = n_ty * n, rounds = (tiles + cap - 1) / cap, cost = rounds * ((L.Lz + n - 1) / n + 2);
    if (best < 0 || cost < best) { best = cost; best_n = n; }
  }
  return best_n;
}

// blocks of one launch (= block partials of the fused measurement); grid_cap = SMs
int sc_ws_blocks(const ScLayout& L, int ZT, int grid_cap, int variant) {
  const int ty = ws_ty(variant);
  const int n_tiles = ((L.Ly + ty - 1) / ty) * sc_ws_chunks(L, ZT, grid_cap, variant);
  const int cap = grid_cap * ws_ctas_per_sm(variant);
  return n_tiles < cap ? n_tiles : cap;
}

cudaError_t launch_sweep_sc_ws(cudaStream_t st, float* s, ScLayout L, int ZT, int grid_cap, int variant, uint32_t* sched, SweepParams p, int colour, Meas m) {
  const int cap = grid_cap * ws_ctas_per_sm(variant);
  int n_zc = sc_ws_chunks(L, ZT, grid_cap, variant);
  if (L.flag_in && n_zc > L.Lz / 2) n_zc = L.Lz / 2 > 0 ? L.Lz / 2 : 1;   // neighbour flags: the boundary chunks hold the planes next to the ghosts
  if (variant == 5) return ws_pick<8, 512, 4, 3>(st, s, L, n_zc, cap, sched, p, colour, m);
  if (variant == 4) return ws_pick<7, 1024, 4, 2>(st, s, L, n_zc, cap, sched, p, colour, m);
  if (variant == 3) return ws_pick<16, 1024, 4, 1>(st, s, L, n_zc, cap, sched, p, colour, m);
  if (variant == 1) return ws_pick<8, 1024, 6, 1>(st, s, L, n_zc, cap, sched, p, colour, m);
  if (variant == 2) return ws_pick<4, 1024, 4, 3>(st, s, L, n_zc, cap, sched, p, colour, m);
  return ws_pick<4, 1024, 5, 2>(st, s, L, n_zc, cap, sched, p, colour, m);
}

// ---- diagnostic: one colour pass of the 7-row kernel with every plane folded onto the first `planes` (a power of two) ----------
cudaError_t launch_sweep_sc_ws_alias(cudaStream_t st, float* s, ScLayout L, int grid_cap, uint32_t* sched, SweepParams p, int colour, int planes) {
  if (!sc_ws_variant_supported(L, 4) || L.ghost || planes < 2 || (planes & (planes - 1)) || planes > L.Lz) return cudaErrorInvalidValue;
  const int cap = grid_cap * ws_ctas_per_sm(4);
  const int n_zc = sc_ws_chunks(L, 0, grid_cap, 4);
  FusedArgs f{0, 0, nullptr};
  f.zmask = (uint32_t)planes - 1u;
  const int aniso = (p.K == 0.0f) ? ANISO_NONE : ((p.ex == 0.0f && p.ey == 0.0f && p.ez == 1.0f) ? ANISO_Z : ANISO_GENERAL);
  const Meas m{nullptr, 0, nullptr};
  switch (aniso) {
    case ANISO_NONE: return ws_go<7, 1024, 4, 2, ANISO_NONE, false, false, false, true>(st, s, L, n_zc, cap, sched, p, colour, m, f);
    case ANISO_Z: return ws_go<7, 1024, 4, 2, ANISO_Z, false, false, false, true>(st, s, L, n_zc, cap, sched, p, colour, m, f);
    default: return ws_go<7, 1024, 4, 2, ANISO_GENERAL, false, false, false, true>(st, s, L, n_zc, cap, sched, p, colour, m, f);
  }
}

// ---- fused launches: n_sweeps whole sweeps (2 n_sweeps colour passes) in ONE launch (variants 2, 4, 5) --------------------
bool sc_ws_fused_supported(const ScLayout& L, int variant) {
  return !L.ghost && (variant == 2 || variant == 4 || variant == 5) && sc_ws_variant_supported(L, variant);
}
// chunks in z of a fused launch: ZT planes each (ZT = 0: 24)
int sc_ws_fused_chunks(const ScLayout& L, int ZT) {
  const int zt = ZT > 0 ? ZT : 24;
  return (L.Lz + zt - 1) / zt;
}
int sc_ws_fused_blocks(const ScLayout& L, int ZT, int grid_cap, int variant, int n_sweeps) {
  const long long n_tiles = (long long)((L.Ly + ws_ty(variant) - 1) / ws_ty(variant)) * sc_ws_fused_chunks(L, ZT) * 2 * n_sweeps;
  const long long cap = (long long)grid_cap * ws_ctas_per_sm(variant);
  return (int)(n_tiles < cap ? n_tiles : cap);
}
cudaError_t launch_sweep_sc_ws_fused(cudaStream_t st, float* s, ScLayout L, int ZT, int lag, int grid_cap, int variant, uint32_t* sched,
                                     uint32_t* done, SweepParams p, int n_sweeps, Meas m) {
  const int n_zc = sc_ws_fused_chunks(L, ZT);
  if (!sc_ws_fused_supported(L, variant) || n_sweeps < 1 || lag < 3 || 2 * n_sweeps * n_zc > kWsDoneWords) return cudaErrorInvalidValue;
  const int cap = grid_cap * ws_ctas_per_sm(variant);
  const FusedArgs f{2 * n_sweeps, lag, done};
  if (variant == 5) return ws_pick<8, 512, 4, 3>(st, s, L, n_zc, cap, sched, p, 0, m, f);
  if (variant == 4) return ws_pick<7, 1024, 4, 2>(st, s, L, n_zc, cap, sched, p, 0, m, f);
  return ws_pick<4, 1024, 4, 3>(st, s, L, n_zc, cap, sched, p, 0, m, f);
}

}  // namespace hb
