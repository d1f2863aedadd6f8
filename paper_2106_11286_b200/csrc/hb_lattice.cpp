// hb_lattice.cpp -- host-side lattice builder and graph colouring.
//
// The paper claims "any crystal lattice" through its linearised spin arrays (PAPER.md lines
// 30, 34) without saying how neighbours are found.  Here a lattice is either implicit
// (Bravais lattice + basis, periodic) or an explicit CSR neighbour table; this file produces
// the tables for bcc, fcc and the free-surface fcc sphere, colours them and validates what
// callers pass in.  Neighbour order is part of the arithmetic contract (include/hb.h).
#include <algorithm>
#include <cmath>

#include "hb_internal.h"

namespace hb {

namespace {

inline int32_t pmod(int32_t a, int32_t m) {
  const int32_t r = a % m;
  return r < 0 ? r + m : r;
}

}  // namespace

// bcc: site b*Nc + cell.  A corner (b = 0) of cell (x,y,z) touches the centres of the eight
// cells (x-1|x, y-1|y, z-1|z); a centre (b = 1) touches the corners of (x|x+1, y|y+1, z|z+1).
void build_bcc_csr(int32_t Lx, int32_t Ly, int32_t Lz, HostCsr& g) {
  const int64_t nc = (int64_t)Lx * Ly * Lz;
  g.n = 2 * nc;
  g.row_ptr.resize(g.n + 1);
  g.col.resize(8 * g.n);
  g.colour.resize(g.n);
  g.n_colours = 2;
  for (int64_t i = 0; i <= g.n; ++i) g.row_ptr[i] = 8 * i;
  for (int32_t b = 0; b < 2; ++b) {
    const int32_t lo = b ? 0 : -1;
    for (int32_t z = 0; z < Lz; ++z)
      for (int32_t y = 0; y < Ly; ++y)
        for (int32_t x = 0; x < Lx; ++x) {
          const int64_t i = b * nc + ((int64_t)z * Ly + y) * Lx + x;
          int32_t* out = &g.col[8 * i];
          for (int32_t s = 0; s < 8; ++s) {          // s = 4*sz + 2*sy + sx, x fastest
            const int32_t cx = pmod(x + lo + (s & 1), Lx);
            const int32_t cy = pmod(y + lo + ((s >> 1) & 1), Ly);
            const int32_t cz = pmod(z + lo + ((s >> 2) & 1), Lz);
            out[s] = (int32_t)((1 - b) * nc + ((int64_t)cz * Ly + cy) * Lx + cx);
          }
          g.colour[i] = b;
        }
  }
}

// fcc: four simple-cubic sublattices; in doubled coordinates a site is 2*(x,y,z) + d_b with
// d_0 = (0,0,0), d_1 = (0,1,1), d_2 = (1,0,1), d_3 = (1,1,0).  The parity pattern of a doubled
// coordinate triple names the sublattice: b = 0 if all even, else the index of the even axis + 1.
void build_fcc_csr(int32_t Lx, int32_t Ly, int32_t Lz, HostCsr& g) {
  static const int8_t off[12][3] = {{1, 1, 0}, {1, -1, 0}, {-1, 1, 0}, {-1, -1, 0}, {1, 0, 1}, {1, 0, -1},
                                    {-1, 0, 1}, {-1, 0, -1}, {0, 1, 1}, {0, 1, -1}, {0, -1, 1}, {0, -1, -1}};
  static const int8_t dbl[4][3] = {{0, 0, 0}, {0, 1, 1}, {1, 0, 1}, {1, 1, 0}};
  const int64_t nc = (int64_t)Lx * Ly * Lz;
  g.n = 4 * nc;
  g.row_ptr.resize(g.n + 1);
  g.col.resize(12 * g.n);
  g.colour.resize(g.n);
  g.n_colours = 4;
  for (int64_t i = 0; i <= g.n; ++i) g.row_ptr[i] = 12 * i;
  for (int32_t b = 0; b < 4; ++b)
    for (int32_t z = 0; z < Lz; ++z)
      for (int32_t y = 0; y < Ly; ++y)
        for (int32_t x = 0; x < Lx; ++x) {
          const int64_t i = b * nc + ((int64_t)z * Ly + y) * Lx + x;
          for (int32_t k = 0; k < 12; ++k) {
            const int32_t X = pmod(2 * x + dbl[b][0] + off[k][0], 2 * Lx);
            const int32_t Y = pmod(2 * y + dbl[b][1] + off[k][1], 2 * Ly);
            const int32_t Z = pmod(2 * z + dbl[b][2] + off[k][2], 2 * Lz);
            const int32_t nb = (X & 1) ? ((Y & 1) ? 3 : 2) : ((Y & 1) ? 1 : 0);
            g.col[12 * i + k] = (int32_t)(nb * nc + ((int64_t)(Z / 2) * Ly + (Y / 2)) * Lx + (X / 2));
          }
          g.colour[i] = b;
        }
}

// Sphere of radius R conventional cells cut from fcc, free surface (A10).
void build_fcc_sphere_csr(int32_t R, HostCsr& g, std::vector<int32_t>& xyz) {
  static const int8_t off[12][3] = {{1, 1, 0}, {1, -1, 0}, {-1, 1, 0}, {-1, -1, 0}, {1, 0, 1}, {1, 0, -1},
                                    {-1, 0, 1}, {-1, 0, -1}, {0, 1, 1}, {0, 1, -1}, {0, -1, 1}, {0, -1, -1}};
  const int32_t D = 2 * R;
  const int64_t W = 2 * (int64_t)D + 3;                // one guard cell on every side
  std::vector<int32_t> id((size_t)(W * W * W), -1);
  auto at = [&](int32_t X, int32_t Y, int32_t Z) -> int32_t& {
    return id[(size_t)(((Z + D + 1) * W + (Y + D + 1)) * W + (X + D + 1))];
  };
  xyz.clear();
  int32_t n = 0;
  for (int32_t Z = -D; Z <= D; ++Z)
    for (int32_t Y = -D; Y <= D; ++Y) {
      const int64_t rem = (int64_t)D * D - (int64_t)Z * Z - (int64_t)Y * Y;
      if (rem < 0) continue;
      for (int32_t X = -D; X <= D; ++X) {
        if (((X ^ Y ^ Z) & 1) || (int64_t)X * X > rem) continue;   // X+Y+Z even and inside
        at(X, Y, Z) = n++;
        xyz.push_back(X); xyz.push_back(Y); xyz.push_back(Z);
      }
    }
  g.n = n;
  g.row_ptr.assign((size_t)n + 1, 0);
  g.col.clear();
  g.col.reserve((size_t)n * 12);
  for (int32_t i = 0; i < n; ++i) {
    const int32_t X = xyz[3 * i], Y = xyz[3 * i + 1], Z = xyz[3 * i + 2];
    for (int32_t k = 0; k < 12; ++k) {
      const int32_t j = at(X + off[k][0], Y + off[k][1], Z + off[k][2]);
      if (j >= 0) g.col.push_back(j);
    }
    g.row_ptr[i + 1] = (int64_t)g.col.size();
  }
  g.colour.assign(n, 0);
  g.n_colours = 0;
}

// Greedy first-fit in site order: the smallest colour not used by an already coloured neighbour.
void greedy_first_fit(HostCsr& g) {
  g.colour.assign(g.n, -1);
  std::vector<int64_t> stamp;                          // stamp[c] == i+1  <=> colour c is taken around i
  int32_t used = 0;
  for (int64_t i = 0; i < g.n; ++i) {
    for (int64_t k = g.row_ptr[i]; k < g.row_ptr[i + 1]; ++k) {
      const int32_t c = g.colour[g.col[k]];
      if (c >= 0) stamp[c] = i + 1;
    }
    int32_t c = 0;
    while (c < used && stamp[c] == i + 1) ++c;
    if (c == used) { stamp.push_back(0); ++used; }
    g.colour[i] = c;
  }
  g.n_colours = used;
}

std::string validate_csr(int64_t n, const int64_t* row_ptr, const int32_t* col, int64_t n_own) {
  if (n_own < 0 || n_own > n) n_own = n;
  if (n < 0 || n > 0xFFFFFFFFll) return "n_sites out of range";
  if (!row_ptr) return "row_ptr is NULL";
  if (row_ptr[0] != 0) return "row_ptr[0] != 0";
  for (int64_t i = 0; i < n; ++i)
    if (row_ptr[i + 1] < row_ptr[i]) return "row_ptr not monotone";
  if (row_ptr[n] >= 0x7FFFFFFFll) return "more than 2^31-2 neighbour entries";
  if (row_ptr[n] > 0 && !col) return "col_idx is NULL";
  for (int64_t i = 0; i < n; ++i)
    for (int64_t k = row_ptr[i]; k < row_ptr[i + 1]; ++k) {
      const int64_t j = col[k];
      if (j < 0 || j >= n) return "col_idx out of range";
      if (j == i) return "self loop";
    }
  for (int64_t i = n_own; i < n; ++i)
    if (row_ptr[i + 1] != row_ptr[i]) return "the row of a ghost site must be empty";
  // symmetric with multiplicity: #(j in row i) == #(i in row j).  Rows of bounded length are compared pair by pair
  // (O(sum of deg^2): lattices); a table with long rows (hubs) compares the sorted lists of (i, j) and (j, i) instead
  int64_t maxdeg = 0;
  for (int64_t i = 0; i < n; ++i) maxdeg = std::max<int64_t>(maxdeg, row_ptr[i + 1] - row_ptr[i]);
  if (maxdeg > 64) {
    std::vector<uint64_t> fwd, rev;
    fwd.reserve((size_t)row_ptr[n]); rev.reserve((size_t)row_ptr[n]);
    for (int64_t i = 0; i < n; ++i)
      for (int64_t k = row_ptr[i]; k < row_ptr[i + 1]; ++k) {
        if (col[k] >= n_own) continue;   // an edge into a ghost site has no counterpart here
        fwd.push_back(((uint64_t)i << 32) | (uint32_t)col[k]);
        rev.push_back(((uint64_t)(uint32_t)col[k] << 32) | (uint64_t)i);
      }
    std::sort(fwd.begin(), fwd.end());
    std::sort(rev.begin(), rev.end());
    return fwd == rev ? "" : "neighbour table is not symmetric";
  }
  for (int64_t i = 0; i < n; ++i)
    for (int64_t k = row_ptr[i]; k < row_ptr[i + 1]; ++k) {
      const int64_t j = col[k];
      if (j >= n_own) continue;   // an edge into a ghost site has no counterpart here
      int64_t a = 0, b = 0;
      for (int64_t q = row_ptr[i]; q < row_ptr[i + 1]; ++q) a += (col[q] == j);
      for (int64_t q = row_ptr[j]; q < row_ptr[j + 1]; ++q) b += (col[q] == i);
      if (a != b) return "neighbour table is not symmetric";
    }
  return "";
}

std::string validate_colouring(int64_t n, const int64_t* row_ptr, const int32_t* col, const int32_t* colour,
                               int32_t n_colours, int64_t n_own) {
  if (n_colours < 1 && n > 0) return "n_colours < 1";
  if (n_own < 0 || n_own > n) n_own = n;
  for (int64_t i = n_own; i < n; ++i)
    if (colour[i] < 0 || colour[i] >= n_colours) return "colour out of range";
  for (int64_t i = 0; i < n_own; ++i) {
    if (colour[i] < 0 || colour[i] >= n_colours) return "colour out of range";
    for (int64_t k = row_ptr[i]; k < row_ptr[i + 1]; ++k)
      if (colour[col[k]] == colour[i]) return "two neighbouring sites share a colour";
  }
  return "";
}

}  // namespace hb
