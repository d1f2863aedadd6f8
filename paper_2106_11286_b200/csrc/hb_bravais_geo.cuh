// hb_bravais_geo.cuh -- compile-time geometry of the periodic Bravais lattices with a basis (bcc, fcc): the neighbour list
// of every sublattice in the order of the arithmetic contract (include/hb.h), shared by hb_bravais.cu and hb_bravais_ws.cu.
#pragma once
#include "hb_internal.h"

namespace hb {
namespace {

struct Nbr { int nb, dx, dy, dz; };

// floor(t / 2) for t in {-1, 0, 1, 2}
__host__ __device__ constexpr int half_floor(int t) { return t < 0 ? -1 : t / 2; }

template <int KIND> struct Geo;

// bcc: a corner (b = 0) of cell (x,y,z) touches the centres of cells (x-1|x, y-1|y, z-1|z), a
// centre (b = 1) the corners of (x|x+1, y|y+1, z|z+1); k = 4 sz + 2 sy + sx, x fastest.
template <> struct Geo<BR_BCC> {
  static constexpr int NB = 2, Z = 8;
  __host__ __device__ static constexpr Nbr nbr(int b, int k) {
    const int lo = b ? 0 : -1;
    return Nbr{1 - b, lo + (k & 1), lo + ((k >> 1) & 1), lo + ((k >> 2) & 1)};
  }
};

// fcc: four sc sublattices; in doubled coordinates a site is 2(x,y,z) + d_b with d_0 = (0,0,0),
// d_1 = (0,1,1), d_2 = (1,0,1), d_3 = (1,1,0); the twelve neighbour offsets in the order of
// include/hb.h.  The parity pattern of the doubled neighbour coordinate names its sublattice.
template <> struct Geo<BR_FCC> {
  static constexpr int NB = 4, Z = 12;
  __host__ __device__ static constexpr Nbr nbr(int b, int k) {
    const int off[12][3] = {{1, 1, 0}, {1, -1, 0}, {-1, 1, 0}, {-1, -1, 0}, {1, 0, 1}, {1, 0, -1},
                            {-1, 0, 1}, {-1, 0, -1}, {0, 1, 1}, {0, 1, -1}, {0, -1, 1}, {0, -1, -1}};
    const int dbl[4][3] = {{0, 0, 0}, {0, 1, 1}, {1, 0, 1}, {1, 1, 0}};
    const int tx = dbl[b][0] + off[k][0], ty = dbl[b][1] + off[k][1], tz = dbl[b][2] + off[k][2];
    const bool ox = (tx & 1) != 0, oy = (ty & 1) != 0;
    return Nbr{ox ? (oy ? 3 : 2) : (oy ? 1 : 0), half_floor(tx), half_floor(ty), half_floor(tz)};
  }
};

// how many of the Z neighbours of sublattice B sit on lower sublattices
template <int KIND, int B>
__host__ __device__ constexpr int n_low() {
  int c = 0;
  for (int k = 0; k < Geo<KIND>::Z; ++k) c += Geo<KIND>::nbr(B, k).nb < B ? 1 : 0;
  return c;
}

// The neighbours of a sublattice sit in a window of two rows and two planes: dy in {lo, lo + 1}, dz in {lo, lo + 1} with
// lo = -1 or 0 (bcc corner: -1, -1; bcc centre: 0, 0; fcc b0 -1, -1; b1 0, 0; b2 -1, 0; b3 0, -1).  axis 1 = y, 2 = z.
template <int KIND>
__host__ __device__ constexpr int window_lo(int b, int axis) {
  int lo = 1;
  for (int k = 0; k < Geo<KIND>::Z; ++k) {
    const Nbr g = Geo<KIND>::nbr(b, k);
    const int d = axis == 1 ? g.dy : g.dz;
    lo = d < lo ? d : lo;
  }
  return lo;
}
template <int KIND>
__host__ __device__ constexpr bool windows_are_two_wide() {
  for (int b = 0; b < Geo<KIND>::NB; ++b)
    for (int k = 0; k < Geo<KIND>::Z; ++k) {
      const Nbr g = Geo<KIND>::nbr(b, k);
      if (g.dy - window_lo<KIND>(b, 1) > 1 || g.dz - window_lo<KIND>(b, 2) > 1 || g.nb == b) return false;
    }
  return true;
}
static_assert(windows_are_two_wide<BR_BCC>() && windows_are_two_wide<BR_FCC>(), "staging windows of hb_bravais_ws.cu");

}  // namespace
}  // namespace hb
