// hb_oracle.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, single-threaded CPU statement of what the hot path of
// arXiv 2106.11286 computes: Metropolis single-spin updates of the classical
// anisotropic Heisenberg model.  Only tests/, __graft_entry__.smoke() and the
// cpu_baseline / --impl reference legs of bench.py may load this file.  It
// shares no code, header, table or constant generator with the CUDA path in
// paper_2106_11286_b200/csrc; every constant below is typed here by hand.
//
// [P:n] = /root/reference/PAPER.md line n.  [D:x] = DESIGN.md reading x.
//
//   eq. (1)  [P:13]   H = -J sum_<ij> S_i.S_j - sum_i K_i (S_i.e_i)^2
//                     (each bond once [D:A1]; nearest neighbours [D:A2];
//                      one (K_i, e_i) per site [D:A11])
//   steps (i)-(iii) [P:20]  pick spin, propose random orientation, accept if
//                     dH <= 0 or P <= exp(-beta dH)
//   eq. (2)  [P:22]   M = (1/N|S|) sum_i S_i , |S| = 1 [P:40]
//   storage  [P:30,50] three linear 4-byte float arrays (x, y, z)
//
// Two programs live here:
//   O32  fp32, colour-ordered sweep, counter-based Philox stream, the
//        arithmetic contract of DESIGN.md section 4 (trajectory oracle).
//   O64  fp64, the paper's steps (i)-(iii) literally: random site choice with
//        std::mt19937_64, libm sin/cos/exp (statistics oracle).
//
// Pins (tests/test_oracle_*.py, all "-m 'not gpu'"): Philox known answers,
// MT19937-64 known answers, sphere map vs the closed form in double, spec
// sincos/exp vs libm, |S|=1, local dH = brute-force difference of total energy,
// single-spin anisotropy closed form, Heisenberg chain closed form, T=inf and
// T->0 limits, sc T_c ~ 1.44, lattice counts vs brute force, checkpoint and
// order invariance.  No function here is "parity unpinned".
//
// Build: g++ -O2 -std=c++17 -ffp-contract=off -fno-fast-math -shared -fPIC
#include <cmath>
#include <cstdint>
#include <cstring>
#include <random>
#include <vector>

namespace {

// ---------------------------------------------------------------------------
// Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11), written from the round
// definition:  (c0,c1,c2,c3) -> (hi(M1*c2)^c1^k0, lo(M1*c2), hi(M0*c0)^c3^k1, lo(M0*c0)),
// key bumped by the Weyl constants after each round; 10 rounds.  [D:4.1]
// ---------------------------------------------------------------------------
void philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
  uint32_t k0 = key[0], k1 = key[1];
  for (int round = 0; round < 10; ++round) {
    const uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
    const uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
    const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
    const uint32_t n1 = (uint32_t)p1;
    const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
    const uint32_t n3 = (uint32_t)p0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += 0x9E3779B9u;
    k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// draw 0 = Metropolis attempt of sweep s at site i ; draw 1 = initial state. [D:4.1]
void philox_site(uint64_t seed, uint32_t site, uint32_t draw, uint64_t sweep, uint32_t out[4]) {
  const uint32_t ctr[4] = {site, draw, (uint32_t)sweep, (uint32_t)(sweep >> 32)};
  const uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
  philox4x32_10(ctr, key, out);
}

// u(r) = (2*(r>>9) + 1) * 2^-24 : odd multiples of 2^-24, exact in fp32,
// strictly inside (0,1), symmetric about 1/2.  "P is a random number between
// 0 and 1" [P:20], open at both ends [D:A5].
uint32_t odd24(uint32_t r) { return 2u * (r >> 9) + 1u; }
float u01(uint32_t r) { return (float)odd24(r) * 5.9604644775390625e-08f; /* 2^-24 */ }

// cos and sin of phi = 2*pi*k/2^24 for odd k in [1, 2^24-1].  [D:4.3]
// Exact integer quadrant reduction, then Taylor polynomials on |t| <= pi/4,
// Horner with fused multiply-adds, coefficients = fp32 roundings of 1/n!.
void sincos_spec(uint32_t k, float* sn, float* cs) {
  const int32_t q = (int32_t)((k + (1u << 21)) >> 22);          // 0..4
  const int32_t rem = (int32_t)k - q * (1 << 22);               // [-2^21, 2^21)
  const float t = (float)rem * 3.74507039e-07f;                 // fp32(pi) * 2^-23
  const float t2 = t * t;
  float ps = 2.75573188e-06f;                                   //  1/362880
  ps = fmaf(ps, t2, -1.98412701e-04f);                          // -1/5040
  ps = fmaf(ps, t2, 8.33333377e-03f);                           //  1/120
  ps = fmaf(ps, t2, -1.66666672e-01f);                          // -1/6
  const float s = fmaf(t * t2, ps, t);
  float pc = 2.48015876e-05f;                                   //  1/40320
  pc = fmaf(pc, t2, -1.38888892e-03f);                          // -1/720
  pc = fmaf(pc, t2, 4.16666679e-02f);                           //  1/24
  pc = fmaf(pc, t2, -0.5f);                                     // -1/2
  const float c = fmaf(t2, pc, 1.0f);
  switch (q & 3) {
    case 0: *cs = c;  *sn = s;  break;
    case 1: *cs = -s; *sn = c;  break;
    case 2: *cs = -c; *sn = -s; break;
    default: *cs = s; *sn = -c; break;
  }
}

// "a new orientation is proposed randomly" [P:20]: uniform on the unit sphere
// [D:A4], Archimedes' map  z = 1-2u1, r = sqrt(1-z^2), phi = 2 pi u2.  [D:4.2]
void sphere(uint32_t r0, uint32_t r1, float out[3]) {
  const float u1 = u01(r0);
  const float z = fmaf(-2.0f, u1, 1.0f);        // exact
  const float rr = sqrtf(fmaf(-z, z, 1.0f));    // IEEE square root
  float sn, cs;
  sincos_spec(odd24(r1), &sn, &cs);
  out[0] = rr * cs;
  out[1] = rr * sn;
  out[2] = z;
}

// exp(x) for x in [-17, 0].  [D:4.5]  Cody-Waite reduction with ln2 split in
// two, degree-7 Taylor polynomial, result scaled by 2^n built from bits.
float exp_spec(float x) {
  const float n = nearbyintf(x * 1.44269502e+00f);  // round half to even
  float r = fmaf(n, -0.693359375f, x);
  r = fmaf(n, 2.12194442e-04f, r);
  float p = 1.98412701e-04f;                         // 1/5040
  p = fmaf(p, r, 1.38888892e-03f);                   // 1/720
  p = fmaf(p, r, 8.33333377e-03f);                   // 1/120
  p = fmaf(p, r, 4.16666679e-02f);                   // 1/24
  p = fmaf(p, r, 1.66666672e-01f);                   // 1/6
  p = fmaf(p, r, 0.5f);
  p = fmaf(p, r, 1.0f);
  p = fmaf(p, r, 1.0f);
  const uint32_t bits = (uint32_t)((int32_t)n + 127) << 23;
  float scale;
  std::memcpy(&scale, &bits, 4);
  return p * scale;
}

// ---------------------------------------------------------------------------
// Lattice = neighbour lists in canonical order + colours + per-site anisotropy.
// The oracle always walks explicit neighbour lists; nothing is implicit.
// ---------------------------------------------------------------------------
struct Lattice {
  int64_t n = 0;
  std::vector<int64_t> row_ptr;   // n+1
  std::vector<int32_t> col;       // nnz, canonical order per row [D:A16]
  std::vector<int32_t> colour;    // n
  int32_t n_colours = 0;
  std::vector<float> K;           // n
  std::vector<float> e;           // 3n, (ex,ey,ez) per site
  std::vector<int32_t> xyz;       // 3n doubled integer coordinates (sphere only)
};

int32_t wrap(int32_t a, int32_t L) { a %= L; return a < 0 ? a + L : a; }

// rows are appended in ascending site id; finish() fills the defaults
void add_row(Lattice& lat, const std::vector<int32_t>& r) {
  if (lat.row_ptr.empty()) lat.row_ptr.push_back(0);
  lat.col.insert(lat.col.end(), r.begin(), r.end());
  lat.row_ptr.push_back((int64_t)lat.col.size());
}
void finish(Lattice& lat) {
  if (lat.row_ptr.empty()) lat.row_ptr.push_back(0);
  lat.n = (int64_t)lat.row_ptr.size() - 1;
  lat.K.assign(lat.n, 0.0f);
  lat.e.assign(3 * lat.n, 0.0f);
  for (int64_t i = 0; i < lat.n; ++i) lat.e[3 * i + 2] = 1.0f;
}

// simple cubic, periodic; id = (z*Ly + y)*Lx + x [D:A15]; neighbours in the
// order -x,+x,-y,+y,-z,+z [D:A16]; colour = (x+y+z) mod 2 (even L) [D:a2].
Lattice* build_sc(int32_t Lx, int32_t Ly, int32_t Lz) {
  auto* lat = new Lattice;
  auto id = [&](int32_t x, int32_t y, int32_t z) {
    return (int32_t)(((int64_t)wrap(z, Lz) * Ly + wrap(y, Ly)) * Lx + wrap(x, Lx));
  };
  for (int32_t z = 0; z < Lz; ++z)
    for (int32_t y = 0; y < Ly; ++y)
      for (int32_t x = 0; x < Lx; ++x) {
        add_row(*lat, {id(x - 1, y, z), id(x + 1, y, z), id(x, y - 1, z),
                       id(x, y + 1, z), id(x, y, z - 1), id(x, y, z + 1)});
        lat->colour.push_back((x + y + z) & 1);
      }
  lat->n_colours = 2;
  finish(*lat);
  return lat;
}

// bcc, periodic, conventional cells; id = b*Nc + cell; b=0 corner (x,y,z),
// b=1 centre (x+1/2,y+1/2,z+1/2).  Corner: centres of cells (x-1|x, y-1|y,
// z-1|z), x fastest; centre: corners of cells (x|x+1, ...). colour = b.
Lattice* build_bcc(int32_t Lx, int32_t Ly, int32_t Lz) {
  auto* lat = new Lattice;
  const int64_t nc = (int64_t)Lx * Ly * Lz;
  auto cell = [&](int32_t x, int32_t y, int32_t z) {
    return ((int64_t)wrap(z, Lz) * Ly + wrap(y, Ly)) * Lx + wrap(x, Lx);
  };
  for (int32_t b = 0; b < 2; ++b)
    for (int32_t z = 0; z < Lz; ++z)
      for (int32_t y = 0; y < Ly; ++y)
        for (int32_t x = 0; x < Lx; ++x) {
          std::vector<int32_t> r;
          if (b == 0) {
            for (int32_t dz = -1; dz <= 0; ++dz)
              for (int32_t dy = -1; dy <= 0; ++dy)
                for (int32_t dx = -1; dx <= 0; ++dx)
                  r.push_back((int32_t)(nc + cell(x + dx, y + dy, z + dz)));
          } else {
            for (int32_t dz = 0; dz <= 1; ++dz)
              for (int32_t dy = 0; dy <= 1; ++dy)
                for (int32_t dx = 0; dx <= 1; ++dx)
                  r.push_back((int32_t)cell(x + dx, y + dy, z + dz));
          }
          add_row(*lat, r);
          lat->colour.push_back(b);
        }
  lat->n_colours = 2;
  finish(*lat);
  return lat;
}

// The 12 fcc nearest-neighbour offsets in doubled integer coordinates [D:A16].
const int32_t FCC_OFF[12][3] = {
    {+1, +1, 0}, {+1, -1, 0}, {-1, +1, 0}, {-1, -1, 0}, {+1, 0, +1}, {+1, 0, -1},
    {-1, 0, +1}, {-1, 0, -1}, {0, +1, +1}, {0, +1, -1}, {0, -1, +1}, {0, -1, -1}};

// fcc, periodic, conventional cells with basis b0 (0,0,0), b1 (0,1/2,1/2),
// b2 (1/2,0,1/2), b3 (1/2,1/2,0); id = b*Nc + cell; colour = b (the four
// simple-cubic sublattices: every nearest neighbour lies in another one).
Lattice* build_fcc(int32_t Lx, int32_t Ly, int32_t Lz) {
  auto* lat = new Lattice;
  const int64_t nc = (int64_t)Lx * Ly * Lz;
  const int32_t basis[4][3] = {{0, 0, 0}, {0, 1, 1}, {1, 0, 1}, {1, 1, 0}};
  auto site = [&](int32_t X, int32_t Y, int32_t Z) {   // doubled coordinates
    X = wrap(X, 2 * Lx); Y = wrap(Y, 2 * Ly); Z = wrap(Z, 2 * Lz);
    const int32_t px = X & 1, py = Y & 1, pz = Z & 1;
    int32_t b = -1;
    for (int32_t k = 0; k < 4; ++k)
      if (basis[k][0] == px && basis[k][1] == py && basis[k][2] == pz) b = k;
    return (int32_t)(b * nc + ((int64_t)(Z >> 1) * Ly + (Y >> 1)) * Lx + (X >> 1));
  };
  for (int32_t b = 0; b < 4; ++b)
    for (int32_t z = 0; z < Lz; ++z)
      for (int32_t y = 0; y < Ly; ++y)
        for (int32_t x = 0; x < Lx; ++x) {
          const int32_t X = 2 * x + basis[b][0], Y = 2 * y + basis[b][1], Z = 2 * z + basis[b][2];
          std::vector<int32_t> r;
          for (const auto& o : FCC_OFF) r.push_back(site(X + o[0], Y + o[1], Z + o[2]));
          add_row(*lat, r);
          lat->colour.push_back(b);
        }
  lat->n_colours = 4;
  finish(*lat);
  return lat;
}

// Sphere cut from fcc, free surface [D:A10]: doubled integer coordinates with
// X+Y+Z even, centre on a site, keep iff X^2+Y^2+Z^2 <= (2R)^2; site order =
// ascending (Z,Y,X); neighbours = the present ones of FCC_OFF in that order.
Lattice* build_fcc_sphere(int32_t R) {
  auto* lat = new Lattice;
  const int32_t D = 2 * R, W = 2 * D + 1;
  std::vector<int32_t> idgrid((size_t)W * W * W, -1);
  auto g = [&](int32_t X, int32_t Y, int32_t Z) -> int32_t& {
    return idgrid[((size_t)(Z + D) * W + (Y + D)) * W + (X + D)];
  };
  int32_t n = 0;
  for (int32_t Z = -D; Z <= D; ++Z)
    for (int32_t Y = -D; Y <= D; ++Y)
      for (int32_t X = -D; X <= D; ++X)
        if (((X + Y + Z) & 1) == 0 && X * X + Y * Y + Z * Z <= D * D) {
          g(X, Y, Z) = n++;
          lat->xyz.push_back(X); lat->xyz.push_back(Y); lat->xyz.push_back(Z);
        }
  for (int32_t i = 0; i < n; ++i) {
    const int32_t X = lat->xyz[3 * i], Y = lat->xyz[3 * i + 1], Z = lat->xyz[3 * i + 2];
    std::vector<int32_t> r;
    for (const auto& o : FCC_OFF) {
      const int32_t A = X + o[0], B = Y + o[1], C = Z + o[2];
      if (A < -D || A > D || B < -D || B > D || C < -D || C > D) continue;
      const int32_t j = g(A, B, C);
      if (j >= 0) r.push_back(j);
    }
    add_row(*lat, r);
  }
  finish(*lat);
  lat->colour.assign(n, 0);
  lat->n_colours = 0;
  return lat;
}

// Greedy first-fit colouring in site order [D:A12].
void greedy_colour(Lattice& lat) {
  lat.colour.assign(lat.n, -1);
  int32_t nc = 0;
  std::vector<char> used;
  for (int64_t i = 0; i < lat.n; ++i) {
    used.assign((size_t)nc + 1, 0);
    for (int64_t k = lat.row_ptr[i]; k < lat.row_ptr[i + 1]; ++k) {
      const int32_t cj = lat.colour[lat.col[k]];
      if (cj >= 0) used[cj] = 1;
    }
    int32_t c = 0;
    while (used[c]) ++c;
    lat.colour[i] = c;
    if (c + 1 > nc) nc = c + 1;
  }
  lat.n_colours = nc;
}

// c5 anisotropy [D:A11]: core sites (12 neighbours) K_core along e_core;
// surface sites (fewer) K_surf along the local radial direction, computed in
// double and rounded to fp32 (z axis for a site at the origin).
void sphere_anisotropy(Lattice& lat, float K_core, const float e_core[3], float K_surf) {
  for (int64_t i = 0; i < lat.n; ++i) {
    const int64_t deg = lat.row_ptr[i + 1] - lat.row_ptr[i];
    if (deg == 12) {
      lat.K[i] = K_core;
      for (int d = 0; d < 3; ++d) lat.e[3 * i + d] = e_core[d];
    } else {
      const double X = lat.xyz[3 * i], Y = lat.xyz[3 * i + 1], Z = lat.xyz[3 * i + 2];
      const double rr = std::sqrt(X * X + Y * Y + Z * Z);
      lat.K[i] = K_surf;
      if (rr > 0.0) {
        lat.e[3 * i] = (float)(X / rr); lat.e[3 * i + 1] = (float)(Y / rr); lat.e[3 * i + 2] = (float)(Z / rr);
      } else {
        lat.e[3 * i] = 0.0f; lat.e[3 * i + 1] = 0.0f; lat.e[3 * i + 2] = 1.0f;
      }
    }
  }
}

// ---------------------------------------------------------------------------
// O32: fp32 colour-ordered sweep with the Philox stream  [D:4]
// ---------------------------------------------------------------------------
struct State32 {
  const Lattice* lat;
  float J;
  uint64_t seed;
  uint64_t sweep = 0;
  uint64_t attempts = 0, accepts = 0;
  std::vector<float> sx, sy, sz;
};

// neighbour field h_i = sum_j S_j, plain fp32 adds in list order
void field32(const State32& st, int64_t i, float h[3]) {
  const Lattice& L = *st.lat;
  float hx = 0.0f, hy = 0.0f, hz = 0.0f;
  for (int64_t k = L.row_ptr[i]; k < L.row_ptr[i + 1]; ++k) {
    const int32_t j = L.col[k];
    hx = hx + st.sx[j]; hy = hy + st.sy[j]; hz = hz + st.sz[j];
  }
  h[0] = hx; h[1] = hy; h[2] = hz;
}

// dH of eq. (1) for S_i -> S' :  -J (S'-S_i).h_i - K_i[(S'.e_i)^2 - (S_i.e_i)^2]
float delta_h32(const State32& st, int64_t i, const float sn[3]) {
  const Lattice& L = *st.lat;
  float h[3];
  field32(st, i, h);
  const float ox = st.sx[i], oy = st.sy[i], oz = st.sz[i];
  const float dx = sn[0] - ox, dy = sn[1] - oy, dz = sn[2] - oz;
  const float dot = fmaf(dz, h[2], fmaf(dy, h[1], dx * h[0]));
  const float ex = L.e[3 * i], ey = L.e[3 * i + 1], ez = L.e[3 * i + 2];
  const float an = fmaf(sn[2], ez, fmaf(sn[1], ey, sn[0] * ex));
  const float ao = fmaf(oz, ez, fmaf(oy, ey, ox * ex));
  return fmaf(-st.J, dot, (-L.K[i]) * ((an - ao) * (an + ao)));
}

// one Metropolis attempt at site i in sweep st.sweep; returns 1 if accepted
int attempt32(State32& st, int64_t i, float beta) {
  uint32_t r[4];
  philox_site(st.seed, (uint32_t)i, 0u, st.sweep, r);
  float sn[3];
  sphere(r[0], r[1], sn);
  const float u3 = u01(r[2]);
  const float dH = delta_h32(st, i, sn);
  bool accept = dH <= 0.0f;
  if (!accept) {
    const float x = (-beta) * dH;
    accept = (x >= -17.0f) && (u3 <= exp_spec(x));
  }
  if (accept) { st.sx[i] = sn[0]; st.sy[i] = sn[1]; st.sz[i] = sn[2]; }
  return accept ? 1 : 0;
}

// order: 0 ascending site id, 1 descending (pin K13: same-colour sites never interact)
void sweep32(State32& st, float T, int order, uint8_t* accept_out) {
  const Lattice& L = *st.lat;
  const float beta = 1.0f / T;
  for (int32_t c = 0; c < L.n_colours; ++c) {
    for (int64_t k = 0; k < L.n; ++k) {
      const int64_t i = order ? L.n - 1 - k : k;
      if (L.colour[i] != c) continue;
      const int a = attempt32(st, i, beta);
      st.attempts += 1; st.accepts += a;
      if (accept_out) accept_out[i] = (uint8_t)a;
    }
  }
  st.sweep += 1;
}

// M = (1/N) sum S_i in double; E: per-site fp32 terms -0.5 J (S_i.h_i) - K_i a_i^2
// summed in double (E32), and the same sum with every product in double (E64).
void measure32(const State32& st, double M[3], double* E32, double* E64) {
  const Lattice& L = *st.lat;
  double mx = 0, my = 0, mz = 0, e32 = 0, e64 = 0;
  for (int64_t i = 0; i < L.n; ++i) {
    mx += (double)st.sx[i]; my += (double)st.sy[i]; mz += (double)st.sz[i];
    float h[3];
    field32(st, i, h);
    const float sh = fmaf(st.sz[i], h[2], fmaf(st.sy[i], h[1], st.sx[i] * h[0]));
    const float a = fmaf(st.sz[i], L.e[3 * i + 2], fmaf(st.sy[i], L.e[3 * i + 1], st.sx[i] * L.e[3 * i]));
    const float term = fmaf(-0.5f * st.J, sh, (-L.K[i]) * (a * a));
    e32 += (double)term;
    double hx = 0, hy = 0, hz = 0;
    for (int64_t k = L.row_ptr[i]; k < L.row_ptr[i + 1]; ++k) {
      const int32_t j = L.col[k];
      hx += (double)st.sx[j]; hy += (double)st.sy[j]; hz += (double)st.sz[j];
    }
    const double ad = (double)st.sx[i] * L.e[3 * i] + (double)st.sy[i] * L.e[3 * i + 1] + (double)st.sz[i] * L.e[3 * i + 2];
    e64 += -0.5 * (double)st.J * ((double)st.sx[i] * hx + (double)st.sy[i] * hy + (double)st.sz[i] * hz)
           - (double)L.K[i] * ad * ad;
  }
  M[0] = mx / (double)L.n; M[1] = my / (double)L.n; M[2] = mz / (double)L.n;
  *E32 = e32; *E64 = e64;
}

// ---------------------------------------------------------------------------
// O64: the paper's steps (i)-(iii) literally, in double  [P:20]
// ---------------------------------------------------------------------------
struct State64 {
  const Lattice* lat;
  double J;
  std::mt19937_64 gen;
  uint64_t attempts = 0, accepts = 0;
  std::vector<double> sx, sy, sz;
};

double uni64(std::mt19937_64& g) { return ((double)(g() >> 11) + 0.5) * (1.0 / 9007199254740992.0); }

void sphere64(std::mt19937_64& g, double s[3]) {
  const double z = 1.0 - 2.0 * uni64(g);
  const double phi = 6.283185307179586476925286766559 * uni64(g);
  const double r = std::sqrt(1.0 - z * z);
  s[0] = r * std::cos(phi); s[1] = r * std::sin(phi); s[2] = z;
}

double site_energy64(const Lattice& L, double J, const std::vector<double>& sx, const std::vector<double>& sy,
                     const std::vector<double>& sz, int64_t i, const double s[3]) {
  double hx = 0, hy = 0, hz = 0;
  for (int64_t k = L.row_ptr[i]; k < L.row_ptr[i + 1]; ++k) {
    const int32_t j = L.col[k];
    hx += sx[j]; hy += sy[j]; hz += sz[j];
  }
  const double a = s[0] * L.e[3 * i] + s[1] * L.e[3 * i + 1] + s[2] * L.e[3 * i + 2];
  return -J * (s[0] * hx + s[1] * hy + s[2] * hz) - (double)L.K[i] * a * a;
}

void sweep64(State64& st, double T) {
  const Lattice& L = *st.lat;
  const double beta = 1.0 / T;
  for (int64_t k = 0; k < L.n; ++k) {
    const int64_t i = (int64_t)(st.gen() % (uint64_t)L.n);      // (i) a spin is chosen at random
    double sn[3];
    sphere64(st.gen, sn);                                        // (ii) new orientation
    const double so[3] = {st.sx[i], st.sy[i], st.sz[i]};
    const double dH = site_energy64(L, st.J, st.sx, st.sy, st.sz, i, sn) -
                      site_energy64(L, st.J, st.sx, st.sy, st.sz, i, so);   // (iii)
    bool accept = dH <= 0.0;
    if (!accept) accept = uni64(st.gen) <= std::exp(-beta * dH);
    st.attempts += 1;
    if (accept) { st.sx[i] = sn[0]; st.sy[i] = sn[1]; st.sz[i] = sn[2]; st.accepts += 1; }
  }
}

// total energy of eq. (1), every directed neighbour entry counted 1/2 [D:A1,A17]
double total_energy64(const Lattice& L, double J, const double* sx, const double* sy, const double* sz) {
  double ex = 0, an = 0;
  for (int64_t i = 0; i < L.n; ++i) {
    for (int64_t k = L.row_ptr[i]; k < L.row_ptr[i + 1]; ++k) {
      const int32_t j = L.col[k];
      ex += sx[i] * sx[j] + sy[i] * sy[j] + sz[i] * sz[j];
    }
    const double a = sx[i] * L.e[3 * i] + sy[i] * L.e[3 * i + 1] + sz[i] * L.e[3 * i + 2];
    an += (double)L.K[i] * a * a;
  }
  return -0.5 * J * ex - an;
}

}  // namespace

// ---------------------------------------------------------------------------
// C entry points (ctypes).  Handles are opaque pointers.
// ---------------------------------------------------------------------------
extern "C" {

void orc_philox4x32_10(const uint32_t* ctr, const uint32_t* key, uint32_t* out) { philox4x32_10(ctr, key, out); }
void orc_philox_site(uint64_t seed, uint32_t site, uint32_t draw, uint64_t sweep, uint32_t* out) {
  philox_site(seed, site, draw, sweep, out);
}
float orc_u01(uint32_t r) { return u01(r); }
void orc_sincos_spec(uint32_t k, float* sn, float* cs) { sincos_spec(k, sn, cs); }
void orc_sincos_spec_batch(uint32_t k0, uint32_t step, int64_t count, float* sn, float* cs) {
  for (int64_t i = 0; i < count; ++i) sincos_spec(k0 + (uint32_t)i * step, sn + i, cs + i);
}
float orc_exp_spec(float x) { return exp_spec(x); }
void orc_exp_spec_batch(const float* x, int64_t count, float* out) {
  for (int64_t i = 0; i < count; ++i) out[i] = exp_spec(x[i]);
}
void orc_sphere(uint32_t r0, uint32_t r1, float* out) { sphere(r0, r1, out); }
void orc_sphere_batch(const uint32_t* r0, const uint32_t* r1, int64_t count, float* out) {
  for (int64_t i = 0; i < count; ++i) sphere(r0[i], r1[i], out + 3 * i);
}
void orc_mt19937_64(uint64_t seed, int64_t count, uint64_t* out) {
  std::mt19937_64 g(seed);
  for (int64_t i = 0; i < count; ++i) out[i] = g();
}

void* orc_lattice_sc(int32_t Lx, int32_t Ly, int32_t Lz) { return build_sc(Lx, Ly, Lz); }
void* orc_lattice_bcc(int32_t Lx, int32_t Ly, int32_t Lz) { return build_bcc(Lx, Ly, Lz); }
void* orc_lattice_fcc(int32_t Lx, int32_t Ly, int32_t Lz) { return build_fcc(Lx, Ly, Lz); }
void* orc_lattice_fcc_sphere(int32_t R) { return build_fcc_sphere(R); }
void* orc_lattice_csr(int64_t n, const int64_t* row_ptr, const int32_t* col, const int32_t* colour, int32_t n_colours) {
  auto* lat = new Lattice;
  lat->n = n;
  lat->row_ptr.assign(row_ptr, row_ptr + n + 1);
  lat->col.assign(col, col + row_ptr[n]);
  lat->K.assign(n, 0.0f);
  lat->e.assign(3 * n, 0.0f);
  for (int64_t i = 0; i < n; ++i) lat->e[3 * i + 2] = 1.0f;
  if (colour) { lat->colour.assign(colour, colour + n); lat->n_colours = n_colours; }
  else greedy_colour(*lat);
  return lat;
}
void orc_lattice_free(void* h) { delete (Lattice*)h; }
void orc_lattice_greedy_colour(void* h) { greedy_colour(*(Lattice*)h); }
void orc_lattice_set_colour(void* h, const int32_t* colour, int32_t n_colours) {
  auto* lat = (Lattice*)h;
  lat->colour.assign(colour, colour + lat->n);
  lat->n_colours = n_colours;
}
void orc_lattice_set_uniform_anisotropy(void* h, float K, const float* e) {
  auto* lat = (Lattice*)h;
  for (int64_t i = 0; i < lat->n; ++i) {
    lat->K[i] = K;
    for (int d = 0; d < 3; ++d) lat->e[3 * i + d] = e[d];
  }
}
void orc_lattice_set_site_anisotropy(void* h, const float* K, const float* e) {
  auto* lat = (Lattice*)h;
  lat->K.assign(K, K + lat->n);
  lat->e.assign(e, e + 3 * lat->n);
}
void orc_lattice_sphere_anisotropy(void* h, float K_core, const float* e_core, float K_surf) {
  sphere_anisotropy(*(Lattice*)h, K_core, e_core, K_surf);
}
int64_t orc_lattice_n(void* h) { return ((Lattice*)h)->n; }
int64_t orc_lattice_nnz(void* h) { return (int64_t)((Lattice*)h)->col.size(); }
int32_t orc_lattice_n_colours(void* h) { return ((Lattice*)h)->n_colours; }
void orc_lattice_get(void* h, int64_t* row_ptr, int32_t* col, int32_t* colour, float* K, float* e, int32_t* xyz) {
  auto* lat = (Lattice*)h;
  if (row_ptr) std::memcpy(row_ptr, lat->row_ptr.data(), sizeof(int64_t) * lat->row_ptr.size());
  if (col) std::memcpy(col, lat->col.data(), sizeof(int32_t) * lat->col.size());
  if (colour) std::memcpy(colour, lat->colour.data(), sizeof(int32_t) * lat->colour.size());
  if (K) std::memcpy(K, lat->K.data(), sizeof(float) * lat->K.size());
  if (e) std::memcpy(e, lat->e.data(), sizeof(float) * lat->e.size());
  if (xyz && !lat->xyz.empty()) std::memcpy(xyz, lat->xyz.data(), sizeof(int32_t) * lat->xyz.size());
}

// ---- O32 ----
void* orc_state32_create(void* lat, float J, uint64_t seed) {
  auto* st = new State32;
  st->lat = (Lattice*)lat; st->J = J; st->seed = seed;
  st->sx.assign(st->lat->n, 0.0f); st->sy.assign(st->lat->n, 0.0f); st->sz.assign(st->lat->n, 1.0f);
  return st;
}
void orc_state32_free(void* h) { delete (State32*)h; }
// a3: S_i = sphere(Philox(site=i, draw=1, sweep=0))
void orc_state32_init_random(void* h) {
  auto* st = (State32*)h;
  for (int64_t i = 0; i < st->lat->n; ++i) {
    uint32_t r[4];
    philox_site(st->seed, (uint32_t)i, 1u, 0u, r);
    float s[3];
    sphere(r[0], r[1], s);
    st->sx[i] = s[0]; st->sy[i] = s[1]; st->sz[i] = s[2];
  }
}
void orc_state32_init_aligned(void* h, const float* dir) {
  auto* st = (State32*)h;
  for (int64_t i = 0; i < st->lat->n; ++i) { st->sx[i] = dir[0]; st->sy[i] = dir[1]; st->sz[i] = dir[2]; }
}
void orc_state32_set(void* h, const float* sx, const float* sy, const float* sz) {
  auto* st = (State32*)h;
  st->sx.assign(sx, sx + st->lat->n); st->sy.assign(sy, sy + st->lat->n); st->sz.assign(sz, sz + st->lat->n);
}
void orc_state32_get(void* h, float* sx, float* sy, float* sz) {
  auto* st = (State32*)h;
  std::memcpy(sx, st->sx.data(), 4 * st->sx.size());
  std::memcpy(sy, st->sy.data(), 4 * st->sy.size());
  std::memcpy(sz, st->sz.data(), 4 * st->sz.size());
}
uint64_t orc_state32_sweep_count(void* h) { return ((State32*)h)->sweep; }
void orc_state32_set_sweep_count(void* h, uint64_t s) { ((State32*)h)->sweep = s; }
void orc_state32_stats(void* h, uint64_t* attempts, uint64_t* accepts) {
  *attempts = ((State32*)h)->attempts; *accepts = ((State32*)h)->accepts;
}
// n sweeps at temperature T.  accept_out: NULL or n*N bytes, [sweep][site].
void orc_state32_sweep(void* h, float T, int64_t n_sweeps, int order, uint8_t* accept_out) {
  auto* st = (State32*)h;
  for (int64_t s = 0; s < n_sweeps; ++s) sweep32(*st, T, order, accept_out ? accept_out + s * st->lat->n : nullptr);
}
void orc_state32_measure(void* h, double* M, double* E32, double* E64) { measure32(*(State32*)h, M, E32, E64); }
// n sweeps, measuring after each: M_out[3n], E_out[n] (E32)
void orc_state32_series(void* h, float T, int64_t n_sweeps, double* M_out, double* E_out) {
  auto* st = (State32*)h;
  for (int64_t s = 0; s < n_sweeps; ++s) {
    sweep32(*st, T, 0, nullptr);
    double e64;
    measure32(*st, M_out + 3 * s, E_out + s, &e64);
  }
}
float orc_state32_delta_h(void* h, int64_t site, const float* s_new) { return delta_h32(*(State32*)h, site, s_new); }
// the proposal and uniform of (site, current sweep) without touching the state
void orc_state32_proposal(void* h, int64_t site, float* s_new, float* u3) {
  auto* st = (State32*)h;
  uint32_t r[4];
  philox_site(st->seed, (uint32_t)site, 0u, st->sweep, r);
  sphere(r[0], r[1], s_new);
  *u3 = u01(r[2]);
}

// ---- O64 ----
void* orc_state64_create(void* lat, double J, uint64_t mt_seed) {
  auto* st = new State64;
  st->lat = (Lattice*)lat; st->J = J; st->gen.seed(mt_seed);
  st->sx.assign(st->lat->n, 0.0); st->sy.assign(st->lat->n, 0.0); st->sz.assign(st->lat->n, 1.0);
  return st;
}
void orc_state64_free(void* h) { delete (State64*)h; }
void orc_state64_init_random(void* h) {
  auto* st = (State64*)h;
  for (int64_t i = 0; i < st->lat->n; ++i) {
    double s[3];
    sphere64(st->gen, s);
    st->sx[i] = s[0]; st->sy[i] = s[1]; st->sz[i] = s[2];
  }
}
void orc_state64_init_aligned(void* h, const double* dir) {
  auto* st = (State64*)h;
  for (int64_t i = 0; i < st->lat->n; ++i) { st->sx[i] = dir[0]; st->sy[i] = dir[1]; st->sz[i] = dir[2]; }
}
void orc_state64_set(void* h, const double* sx, const double* sy, const double* sz) {
  auto* st = (State64*)h;
  st->sx.assign(sx, sx + st->lat->n); st->sy.assign(sy, sy + st->lat->n); st->sz.assign(sz, sz + st->lat->n);
}
void orc_state64_get(void* h, double* sx, double* sy, double* sz) {
  auto* st = (State64*)h;
  std::memcpy(sx, st->sx.data(), 8 * st->sx.size());
  std::memcpy(sy, st->sy.data(), 8 * st->sy.size());
  std::memcpy(sz, st->sz.data(), 8 * st->sz.size());
}
void orc_state64_sweep(void* h, double T, int64_t n_sweeps) {
  for (int64_t s = 0; s < n_sweeps; ++s) sweep64(*(State64*)h, T);
}
void orc_state64_stats(void* h, uint64_t* attempts, uint64_t* accepts) {
  *attempts = ((State64*)h)->attempts; *accepts = ((State64*)h)->accepts;
}
void orc_state64_measure(void* h, double* M, double* E) {
  auto* st = (State64*)h;
  const Lattice& L = *st->lat;
  double mx = 0, my = 0, mz = 0;
  for (int64_t i = 0; i < L.n; ++i) { mx += st->sx[i]; my += st->sy[i]; mz += st->sz[i]; }
  M[0] = mx / (double)L.n; M[1] = my / (double)L.n; M[2] = mz / (double)L.n;
  *E = total_energy64(L, st->J, st->sx.data(), st->sy.data(), st->sz.data());
}
// n sweeps, after each: |M|, E, and mean over sites of (S.e)^2
void orc_state64_series(void* h, double T, int64_t n_sweeps, double* absM, double* E, double* a2) {
  auto* st = (State64*)h;
  const Lattice& L = *st->lat;
  for (int64_t s = 0; s < n_sweeps; ++s) {
    sweep64(*st, T);
    double M[3];
    orc_state64_measure(h, M, E + s);
    absM[s] = std::sqrt(M[0] * M[0] + M[1] * M[1] + M[2] * M[2]);
    double acc = 0;
    for (int64_t i = 0; i < L.n; ++i) {
      const double a = st->sx[i] * L.e[3 * i] + st->sy[i] * L.e[3 * i + 1] + st->sz[i] * L.e[3 * i + 2];
      acc += a * a;
    }
    a2[s] = acc / (double)L.n;
  }
}
double orc_total_energy64(void* lat, double J, const double* sx, const double* sy, const double* sz) {
  return total_energy64(*(Lattice*)lat, J, sx, sy, sz);
}
double orc_state64_delta_h(void* h, int64_t i, const double* s_new) {
  auto* st = (State64*)h;
  const double so[3] = {st->sx[i], st->sy[i], st->sz[i]};
  return site_energy64(*st->lat, st->J, st->sx, st->sy, st->sz, i, s_new) -
         site_energy64(*st->lat, st->J, st->sx, st->sy, st->sz, i, so);
}

}  // extern "C"
