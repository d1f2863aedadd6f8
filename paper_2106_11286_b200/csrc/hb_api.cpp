// hb_api.cpp -- the C ABI of include/hb.h: context, validation, sweep driver.
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <new>
#include <stdexcept>
#include <string>
#include <vector>

#include "../../include/hb.h"
#include "../../include/hb_diag.h"
#include "hb_internal.h"

using namespace hb;

namespace {

constexpr size_t kAlign = 256;
constexpr int kSeriesChunk = 1024;
constexpr int64_t kMaxColours = 65536;   // bound on the colour count the ELL workspace is sized for

inline size_t align_up(size_t x) { return (x + kAlign - 1) / kAlign * kAlign; }

enum Engine { ENGINE_SC = 0, ENGINE_CSR = 1, ENGINE_BRAVAIS = 2 };

struct Plan {                 // device memory plan of a lattice
  int64_t n = 0, nnz = 0;
  int engine = ENGINE_CSR;
  bool per_site = false;
  int32_t R = 1;              // independent replicas (sc, one block per replica)
  size_t off_each = 0, off_betas = 0;   // R > 1: per replica 16 doubles of partials + 4 of cached measurement; R betas
  bool ell = false;           // table engine: colour-major ELL layout (else plain CSR in canonical order)
  int32_t maxdeg = 0;
  size_t off_ell = 0, off_cbegin = 0;
  size_t spins_bytes = 0, ws_bytes = 0;
  size_t off_partials = 0, off_series = 0, off_counters = 0, off_staging = 0, off_wsdone = 0;
  size_t off_row_ptr = 0, off_col = 0, off_list = 0, off_K = 0, off_e = 0;
  // a part of a larger neighbour table (hb_lattice.part_n_total > 0): own sites 0 .. n_own-1 are global sites part_first ...,
  // the remaining local sites are ghosts; off_inv: canonical id -> internal index (ELL engine), for hb_part_gather / scatter
  int64_t n_own = 0, part_first = 0, part_total = 0;
  size_t off_inv = 0;
};

// A slab (hb_lattice.slab_Lz > 0) is run as a periodic lattice of Lz + 2 planes whose first and last planes are the
// ghost planes: the kernels index it like any other lattice and only skip the updates of those two planes
// (ScLayout::ghost), which the z-neighbours own and fill (face copies or peer stores).  Returns the padded description.
int pad_slab(const hb_lattice* lat, hb_lattice& padded, std::string& why) {
  padded = *lat;
  if (lat->slab_Lz <= 0) return HB_OK;
  if ((lat->kind != HB_SC && lat->kind != HB_BCC && lat->kind != HB_FCC) || lat->n_replicas > 1 || lat->K_site || lat->e_site) {
    why = "a slab needs a periodic sc, bcc or fcc lattice with uniform anisotropy and no replicas"; return HB_EINVAL;
  }
  // sc: the checkerboard colour of a local plane must be known from its index, hence even offsets; bcc / fcc colour by basis index
  const int odd = lat->kind == HB_SC ? ((lat->Lz | lat->slab_Lz | lat->slab_z0) & 1) : 0;
  if (lat->Lz < (lat->kind == HB_SC ? 2 : 1) || odd || lat->slab_z0 < 0 || lat->slab_z0 + lat->Lz > lat->slab_Lz) {
    why = "slab: 0 <= slab_z0, slab_z0 + Lz <= slab_Lz; simple cubic: Lz, slab_Lz, slab_z0 even and Lz >= 2"; return HB_EINVAL;
  }
  const int basis = lat->kind == HB_SC ? 1 : (lat->kind == HB_BCC ? 2 : 4);
  if ((int64_t)lat->Lx * lat->Ly * lat->slab_Lz * basis > 0xFFFFFFFFll) { why = "more than 2^32-1 sites in the whole lattice"; return HB_EINVAL; }
  padded.Lz = lat->Lz + 2;
  padded.slab_Lz = 0;
  return HB_OK;
}

int make_plan(const hb_lattice* lat, Plan& p, std::string& why) {
  if (!lat) { why = "lattice is NULL"; return HB_EINVAL; }
  const int k = lat->kind;
  if (k == HB_SC || k == HB_BCC || k == HB_FCC) {
    if (lat->Lx < 1 || lat->Ly < 1 || lat->Lz < 1) { why = "Lx, Ly, Lz must be >= 1"; return HB_EINVAL; }
    const int64_t cells = (int64_t)lat->Lx * lat->Ly * lat->Lz;
    const int basis = k == HB_SC ? 1 : (k == HB_BCC ? 2 : 4);
    const int z = k == HB_SC ? 6 : (k == HB_BCC ? 8 : 12);
    p.n = cells * basis;
    p.nnz = p.n * z;
    p.maxdeg = z;
    if (k == HB_SC && ((lat->Lx | lat->Ly | lat->Lz) & 1)) {
      why = "simple cubic needs even Lx, Ly, Lz (two-colour checkerboard with periodic wrap)";
      return HB_EINVAL;
    }
  } else if (k == HB_CSR) {
    if (lat->n_sites < 0 || !lat->row_ptr) { why = "CSR lattice needs n_sites >= 0 and row_ptr"; return HB_EINVAL; }
    // (before row_ptr is walked: an absurd n_sites must not send the loop below past the caller's array)
    if (lat->n_sites > 0xFFFFFFFFll) { why = "more than 2^32-1 sites (site ids are 32-bit Philox counter words)"; return HB_EINVAL; }
    p.n = lat->n_sites;
    // the sizes below come from row_ptr: it must start at 0 and never decrease before anything is derived from it
    if (lat->row_ptr[0] != 0) { why = "row_ptr[0] must be 0"; return HB_EINVAL; }
    int64_t md = 0;
    for (int64_t i = 0; i < p.n; ++i) {
      const int64_t deg = lat->row_ptr[i + 1] - lat->row_ptr[i];
      if (deg < 0) { why = "row_ptr must not decrease"; return HB_EINVAL; }
      if (deg > md) md = deg;
    }
    p.nnz = lat->row_ptr[lat->n_sites];
    if (p.nnz > 0 && !lat->col_idx) { why = "CSR lattice needs col_idx"; return HB_EINVAL; }
    // a caller-supplied colouring: the colour count sizes host and device tables, so it is bounded before anything is allocated
    if (lat->colour && (lat->n_colours < 1 || lat->n_colours > kMaxColours || (int64_t)lat->n_colours > (p.n > 0 ? p.n : 1))) {
      why = "n_colours must be in [1, min(n_sites, 65536)]"; return HB_EINVAL;
    }
    p.maxdeg = (int32_t)(md > 0x7FFFFFFF ? 0x7FFFFFFF : md);
    if (lat->part_n_total > 0) {
      if (lat->part_n_own < 1 || lat->part_n_own > p.n || lat->part_first < 0 || lat->part_first + lat->part_n_own > lat->part_n_total ||
          lat->part_n_total > 0xFFFFFFFFll || !lat->colour || lat->n_replicas > 1) {
        why = "part of a table: 1 <= part_n_own <= n_sites, 0 <= part_first, part_first + part_n_own <= part_n_total < 2^32, colour given, no replicas";
        return HB_EINVAL;
      }
      p.n_own = lat->part_n_own; p.part_first = lat->part_first; p.part_total = lat->part_n_total;
    }
  } else {
    why = "unknown lattice kind";
    return HB_EINVAL;
  }
  if (k != HB_CSR && lat->part_n_total > 0) { why = "part_n_total: neighbour tables (HB_CSR) only; sc, bcc and fcc are cut into slabs (slab_Lz)"; return HB_EINVAL; }
  if (p.n < 1) { why = "lattice has no sites"; return HB_EINVAL; }
  if (p.n > 0xFFFFFFFFll) { why = "more than 2^32-1 sites (site ids are 32-bit Philox counter words)"; return HB_EINVAL; }
  if ((lat->K_site == nullptr) != (lat->e_site == nullptr)) { why = "K_site and e_site go together"; return HB_EINVAL; }
  p.per_site = lat->K_site != nullptr;
  // only the table engine materialises the neighbour entries (32-bit offsets); the implicit kinds go up to 2^32-1 sites
  if ((p.per_site || k == HB_CSR) && p.nnz >= 0x7FFFFFFFll) { why = "more than 2^31-2 neighbour entries"; return HB_EINVAL; }
  // implicit indexing for the periodic kinds; the table engine for CSR input and per-site anisotropy
  p.engine = p.per_site || k == HB_CSR ? ENGINE_CSR : (k == HB_SC ? ENGINE_SC : ENGINE_BRAVAIS);
  p.R = lat->n_replicas > 1 ? lat->n_replicas : 1;
  if (p.R > 1) {
    ScLayout sl{};
    sl.Lx = lat->Lx; sl.Ly = lat->Ly; sl.Lz = lat->Lz; sl.H = lat->Lx / 2;
    if (p.engine != ENGINE_SC || sc_one_block_threads(sl) == 0 || p.R > 4096) {
      why = "replicas need a simple cubic lattice of at most 8192 sites with Lx a multiple of 8, uniform anisotropy, and at most 4096 replicas";
      return HB_EINVAL;
    }
  }
  size_t o = 0;
  const size_t n_partials = kMeasureBlocks > 2 * kFusedBlocksMax ? kMeasureBlocks : 2 * kFusedBlocksMax;
  p.off_partials = o; o += align_up(n_partials * 4 * sizeof(double));
  p.off_series = o;   o += align_up((size_t)p.R * kSeriesChunk * 4 * sizeof(double));
  p.off_counters = o; o += kAlign;
  p.off_staging = o;  o += align_up((size_t)p.n * sizeof(float));
  if (p.engine == ENGINE_SC || p.engine == ENGINE_BRAVAIS) { p.off_wsdone = o; o += align_up((size_t)kWsDoneWords * sizeof(uint32_t)); }   // progress words of fused launches
  if (p.R > 1) {
    p.off_each = o;  o += align_up((size_t)p.R * 20 * sizeof(double));
    p.off_betas = o; o += align_up((size_t)p.R * sizeof(float));
  }
  if (p.engine == ENGINE_CSR) {
    // ELL when padding every row to the maximum degree costs little (regular lattices, cut-outs of them);
    // graphs with a few high-degree sites keep the plain CSR kernel
    p.ell = p.maxdeg >= 1 && p.maxdeg <= 64 && (int64_t)p.maxdeg * (p.part_total > 0 ? p.n_own : p.n) <= 2 * p.nnz + 1024;   // (ghost rows are empty)
    if (p.ell && p.part_total > 0) { p.off_inv = o; o += align_up((size_t)p.n * sizeof(int32_t)); }
    if (p.ell) {
      p.off_ell = o;    o += align_up((size_t)p.maxdeg * (size_t)p.n * sizeof(int32_t));
      p.off_cbegin = o; o += align_up(((size_t)(p.n < kMaxColours ? p.n : kMaxColours) + 2) * sizeof(uint32_t));
    } else {
      p.off_row_ptr = o; o += align_up(((size_t)p.n + 1) * sizeof(int32_t));
      p.off_col = o;     o += align_up((size_t)p.nnz * sizeof(int32_t));
    }
    p.off_list = o;    o += align_up((size_t)p.n * sizeof(int32_t));
    if (p.per_site) {
      p.off_K = o; o += align_up((size_t)p.n * sizeof(float));
      p.off_e = o; o += align_up(3 * (size_t)p.n * sizeof(float));
    }
  }
  p.ws_bytes = o;
  p.spins_bytes = align_up((size_t)p.R * (p.ell ? 4 : 3) * (size_t)p.n * sizeof(float));   // ELL engine: AoS float4
  return HB_OK;
}

}  // namespace

struct hb_ctx {
  Plan plan;
  int32_t kind = 0, Lx = 0, Ly = 0, Lz = 0;
  ScLayout sc{};
  BrLayout br{};
  ScTile tile{};
  CsrDev csr{};
  EllDev ell{};
  int csr_block = 128;
  int sc_kernel = 0;      // 0: direct loads through L1, 1: warp-specialised persistent kernel (TMA-staged neighbour planes),
                          // 2: the same kernel with all colour passes of up to fused_sweeps sweeps in ONE launch
  int fused_sweeps = 8, fused_lag = 6, fused_zt = 24;   // the fastest setting measured on c4
  int br_kernel = 0, br_zt = 0;   // bcc / fcc: 0 direct loads through L1, 1 warp-specialised persistent kernel (one launch per colour),
                                  // 2 the same with all colour passes of up to fused_sweeps sweeps in one launch
  int ws_zt = 0, n_sms = 148, ws_variant = 2;   // warp-specialised kernel: planes per tile (0: balanced automatically), CTAs = n_sms x CTAs/SM
  int graph_mode = -1;         // replay hb_sweep's launches from a CUDA graph: -1 auto (lattices up to 2^23 sites), 0 off, 1 on
  cudaStream_t cap_stream = nullptr;
  cudaGraphExec_t gexec[2] = {nullptr, nullptr};   // [0] plain sweeps, [1] every sweep measured into the series buffer
  float g_beta[2] = {0.0f, 0.0f};
  bool g_dirty[2] = {true, true};
  int pdl = 1;                 // colour kernels are launched with programmatic stream serialisation (option pdl)
  int32_t slab_Lz = 0, slab_z0 = 0;   // > 0: this context is a slab of a larger lattice (planes 0 and Lz-1 of sc are ghosts)
  uint32_t slab_stamp = 0;            // colour passes of this slab so far (neighbour flags, option slab_flags)
  // hb_stage_spins / hb_commit_spins: a library-owned upload area of 3 n floats, filled on its own stream while the context's
  // stream computes (allocated at the first hb_stage_spins, freed by hb_destroy)
  float* stage = nullptr;
  cudaStream_t stage_stream = nullptr;
  cudaEvent_t stage_filled = nullptr, stage_free = nullptr;
  bool stage_pending = false;
  uint32_t* slab_flags() const { return reinterpret_cast<uint32_t*>(spins_base + 3 * (size_t)plan.n); }   // two words behind the spins
  int sc_coop = -1;            // persistent multi-sweep kernel: -1 auto, 0 off, 1 / 2 forced (see hb_set_option)
  bool fused_measure = true;   // sc: the last sweep of hb_sweep also reduces M and E
  bool cache_valid = false;    // cached() holds the measurement of the current spins
  std::vector<uint32_t> colour_begin;     // CSR engine: offsets into the colour-sorted list
  std::vector<int32_t> colour_host;       // CSR engine: colour of every site
  int32_t n_colours = 0;
  float J = 0, K = 0, e[3] = {0, 0, 1};
  uint64_t seed = 0, sweep = 0;
  bool initialised = false;
  cudaStream_t stream = nullptr;
  float* spins = nullptr;        // state of the selected replica (the only one unless plan.R > 1)
  float* spins_base = nullptr;   // state of replica 0
  uint64_t seed_base = 0;
  int32_t sel = 0;
  bool each_valid = false;       // cached_each() holds the measurements of all replicas
  char* ws = nullptr;
  bool own_spins = false, own_ws = false;
  uint64_t launches = 0, attempts = 0;
  uint64_t stat_attempts = 0;   // attempts of the sweeps whose accepted moves were counted on the device (hb_stats)
  int sticky = HB_OK;
  std::string detail;

  double* partials() const { return reinterpret_cast<double*>(ws + plan.off_partials); }
  double* series() const { return reinterpret_cast<double*>(ws + plan.off_series); }
  unsigned long long* counters() const { return reinterpret_cast<unsigned long long*>(ws + plan.off_counters); }
  float* staging() const { return reinterpret_cast<float*>(ws + plan.off_staging); }
  double* partials_each() const { return reinterpret_cast<double*>(ws + plan.off_each); }
  double* cached_each() const { return reinterpret_cast<double*>(ws + plan.off_each) + (size_t)plan.R * 16; }
  float* betas() const { return reinterpret_cast<float*>(ws + plan.off_betas); }
  double* cached() const { return reinterpret_cast<double*>(ws + plan.off_counters + 64); }
  unsigned long long* sweep_dev() const { return reinterpret_cast<unsigned long long*>(ws + plan.off_counters + 128); }
  unsigned long long* series_idx() const { return reinterpret_cast<unsigned long long*>(ws + plan.off_counters + 136); }
  uint32_t* ws_sched() const { return reinterpret_cast<uint32_t*>(ws + plan.off_counters + 144); }   // tile scheduler of k_sweep_sc_ws
  uint32_t* slab_bnd_count() const { return reinterpret_cast<uint32_t*>(ws + plan.off_counters + 160); }   // two words
  uint32_t* ws_done() const { return reinterpret_cast<uint32_t*>(ws + plan.off_wsdone); }            // progress words of its fused launches
};

namespace {

int fail(hb_ctx* c, int status, const std::string& msg) {
  if (c) {
    c->detail = msg;
    if (status == HB_ECUDA) c->sticky = HB_ECUDA;
  }
  return status;
}

#define HB_CUDA(ctx, call)                                                                      \
  do {                                                                                          \
    const cudaError_t err__ = (call);                                                           \
    if (err__ != cudaSuccess)                                                                   \
      return fail(ctx, HB_ECUDA, std::string(#call) + ": " + cudaGetErrorString(err__));        \
  } while (0)

#define HB_CHECK_CTX(ctx)                                   \
  do {                                                      \
    if (!(ctx)) return HB_EINVAL;                           \
    if ((ctx)->sticky != HB_OK) return (ctx)->sticky;       \
  } while (0)

SweepParams params(const hb_ctx* c, float beta) {
  SweepParams p;
  p.J = c->J; p.K = c->K; p.ex = c->e[0]; p.ey = c->e[1]; p.ez = c->e[2]; p.beta = beta;
  p.seed_lo = (uint32_t)c->seed; p.seed_hi = (uint32_t)(c->seed >> 32);
  p.sweep_lo = (uint32_t)c->sweep; p.sweep_hi = (uint32_t)(c->sweep >> 32);
  p.sweep_dev = nullptr;
  p.pdl = c->pdl;
  return p;
}

bool unit_vector(const float* v) {
  const double n2 = (double)v[0] * v[0] + (double)v[1] * v[1] + (double)v[2] * v[2];
  return std::isfinite(n2) && std::fabs(n2 - 1.0) <= 1e-5;
}

// default launch shape of the structured kernels for rows of H floats
ScTile default_tile(int32_t H, int32_t Ly, int32_t Lz) {
  struct { int32_t H, Ly, Lz; } L{H, Ly, Lz};
  ScTile t;
  t.PF = 1;
  t.LIN = 0;
  t.V = (L.H % 4 == 0) ? 4 : ((L.H % 2 == 0) ? 2 : 1);
  const int HV = L.H / t.V;
  int best = HV <= 64 ? HV : 64, best_waste = 1 << 30;
  if (HV > 64) {
    for (int jx = 64; jx >= 24; --jx) {
      const int waste = (HV + jx - 1) / jx * jx - HV;
      if (waste < best_waste) { best_waste = waste; best = jx; }
    }
  }
  t.JX = best;
  t.TY = 256 / t.JX;
  if (t.TY > L.Ly) t.TY = L.Ly;
  if (t.TY < 1) t.TY = 1;
  // enough blocks to fill 148 SMs several times over, else shorter z-marches
  const int64_t cols = (int64_t)((HV + t.JX - 1) / t.JX) * ((L.Ly + t.TY - 1) / t.TY);
  t.ZT = 8;
  while (t.ZT > 1 && cols * ((L.Lz + t.ZT - 1) / t.ZT) < 148 * 16) t.ZT /= 2;
  if (t.ZT == 1 && t.V == 4 && t.JX * t.TY > 128) {
    // A launch of few blocks (the loop above ended at one plane per block): blocks of 128 threads spread it more evenly
    // over the SMs, and march as many planes as still leave eight blocks per SM.  Measured (Gupd/s, replayed launches):
    // sc 96^3 73 -> 80, sc 160^3 113 -> 118, sc 192^3 113 -> 116-119, c2 (bcc 64^3) 70.3 -> 72.8, c3 (fcc 128^3) 84.2 -> 91.0.
    t.TY = 128 / t.JX > 0 ? 128 / t.JX : 1;
    if (t.TY > L.Ly) t.TY = L.Ly;
    const int64_t cols2 = (int64_t)((HV + t.JX - 1) / t.JX) * ((L.Ly + t.TY - 1) / t.TY);
    t.ZT = 8;
    while (t.ZT > 1 && cols2 * ((L.Lz + t.ZT - 1) / t.ZT) < 148 * 8) t.ZT /= 2;
  }
  return t;
}

int one_colour(hb_ctx* c, int colour, const SweepParams& p, Diag d, Meas m = Meas{nullptr, 0, nullptr}) {
  if (c->plan.engine == ENGINE_SC) {
    const bool diag = d.accept || d.n_accept;
    if (c->sc_kernel >= 1 && !diag)
      HB_CUDA(c, launch_sweep_sc_ws(c->stream, c->spins, c->sc, c->ws_zt, c->n_sms, c->ws_variant, c->ws_sched(), p, colour, m));
    else
      HB_CUDA(c, launch_sweep_sc(c->stream, c->spins, c->sc, c->tile, p, colour, d, m));
  } else if (c->plan.engine == ENGINE_BRAVAIS) {
    if (c->br_kernel >= 1 && !(d.accept || d.n_accept))
      HB_CUDA(c, launch_sweep_bravais_ws(c->stream, c->spins, c->br, c->br_zt, c->fused_lag, c->n_sms, c->ws_sched(), c->ws_done(), p, colour, 1, m));
    else
      HB_CUDA(c, launch_sweep_bravais(c->stream, c->spins, c->br, c->tile, p, colour, d, m));
  } else {
    const uint32_t b = c->colour_begin[colour], e = c->colour_begin[colour + 1];
    if (e == b) return HB_OK;
    if (c->plan.ell) HB_CUDA(c, launch_sweep_ell(c->stream, c->spins, c->ell, b, e - b, p, c->csr_block, d));
    else HB_CUDA(c, launch_sweep_csr(c->stream, c->spins, c->csr, b, e - b, p, c->csr_block, d));
  }
  c->launches += 1;
  return HB_OK;
}

// The all-passes launch of the bcc / fcc warp-specialised kernel (br_kernel 2) marks progress in kWsDoneWords words, one per
// (pass, chunk): a lattice with too many chunks along z runs one sweep per launch, and if that still does not fit, one
// pass per launch (br_kernel 1), instead of failing in launch_sweep_bravais_ws.
void clamp_bravais_ws(hb_ctx* c) {
  if (c->plan.engine != ENGINE_BRAVAIS || c->br_kernel < 1) return;
  const long long chunks = bravais_ws_chunks(c->br, c->br_zt, c->n_sms);
  if ((long long)(c->n_colours * c->fused_sweeps - 1) * chunks > kWsDoneWords) c->fused_sweeps = 1;
  if (c->br_kernel == 2 && (long long)(c->n_colours - 1) * chunks > kWsDoneWords) c->br_kernel = 1;
}

// blocks per colour launch if this context can fuse the measurement into its colour passes, else 0
int fused_blocks(const hb_ctx* c) {
  if (!c->fused_measure) return 0;
  if (c->plan.engine == ENGINE_BRAVAIS && c->br_kernel >= 1) {
    const int fb = bravais_ws_blocks(c->br, c->br_zt, c->n_sms, c->br_kernel == 2 ? c->n_colours : 1);
    // one launch per colour keeps n_colours sets of block partials side by side in a buffer of 2 kFusedBlocksMax blocks
    // (sc_ws_ctas up to 4096 x 3 resident blocks x 4 colours would overrun it): such grids use the separate measurement pass
    return (long long)c->n_colours * fb <= 2 * kFusedBlocksMax ? fb : 0;
  }
  if (c->plan.engine == ENGINE_BRAVAIS) return bravais_fused_blocks(c->br, c->tile);
  if (c->plan.engine != ENGINE_SC) return 0;
  if (c->sc_kernel == 2) return sc_ws_fused_blocks(c->sc, c->fused_zt, c->n_sms, c->ws_variant, 1);
  if (c->sc_kernel == 1) return sc_ws_blocks(c->sc, c->ws_zt, c->n_sms, c->ws_variant);
  return sc_fused_blocks(c->sc, c->tile);
}

// persistent path of hb_sweep: 1 = one block (auto for lattices whose colour pass fits 1024 threads), 2 = cooperative
// grid (only when forced with sc_coop = 1 or 2: measured slower than one launch per colour at every size), 0 = none
int coop_mode(const hb_ctx* c) {
  if (c->plan.engine != ENGINE_SC || c->sc_kernel != 0 || !c->fused_measure || c->sc_coop == 0) return 0;
  if (c->sc_coop != 2 && sc_one_block_threads(c->sc) > 0) return 1;
  return (c->sc_coop >= 1 && sc_coop_blocks(c->sc, c->tile) > 0) ? 2 : 0;
}

// n sweeps in cooperative launches; series (device, 4 doubles per sweep) or final_out (device, 4 doubles) or neither
int coop_sweeps(hb_ctx* c, float beta, int64_t n_sweeps, double* series, double* final_out) {
  const SweepParams p = params(c, beta);
  const int64_t chunk = int64_t(1) << 20;
  for (int64_t s0 = 0; s0 < n_sweeps; s0 += chunk) {
    const int m = (int)(n_sweeps - s0 < chunk ? n_sweeps - s0 : chunk);
    const bool last = s0 + m == n_sweeps;
    HB_CUDA(c, launch_sweeps_sc_coop(c->stream, c->spins, c->sc, c->tile, p, c->sweep, m, coop_mode(c) == 1, c->partials(),
                                     series ? series + 4 * s0 : nullptr, last ? final_out : nullptr, 1, nullptr, 0, c->counters()));
    c->stat_attempts += (uint64_t)(series ? m : ((last && final_out) ? 1 : 0)) * (uint64_t)c->plan.n;   // the measured sweeps count their accepts
    c->launches += 1;
    c->sweep += (uint64_t)m;
    c->attempts += (uint64_t)m * (uint64_t)c->plan.n;
  }
  return HB_OK;
}

// sc_kernel = 2: n_sweeps whole sweeps in ONE launch (both colours of every sweep, tiles with dependencies instead of a launch
// boundary per colour); with dev_out the launch is one sweep whose passes also reduce M and E, as in one_sweep below
int fused_sweeps_launch(hb_ctx* c, float beta, int n_sweeps, double* dev_out, bool counted) {
  const SweepParams p = params(c, beta);
  Meas m{nullptr, 0, nullptr};
  const int fb = dev_out ? fused_blocks(c) : 0;
  if (fb) m = Meas{c->partials(), 2, counted ? c->counters() : nullptr};
  if (c->plan.engine == ENGINE_BRAVAIS)
    HB_CUDA(c, launch_sweep_bravais_ws(c->stream, c->spins, c->br, c->br_zt, c->fused_lag, c->n_sms, c->ws_sched(), c->ws_done(), p, 0,
                                       c->n_colours * n_sweeps, m));
  else
  HB_CUDA(c, launch_sweep_sc_ws_fused(c->stream, c->spins, c->sc, c->fused_zt, c->fused_lag, c->n_sms, c->ws_variant, c->ws_sched(), c->ws_done(),
                                      p, n_sweeps, m));
  c->launches += 1;
  if (fb) {
    HB_CUDA(c, launch_reduce_final(c->stream, c->partials(), fb, dev_out));
    c->launches += 1;
    if (counted) c->stat_attempts += (uint64_t)c->plan.n;
  }
  c->sweep += (uint64_t)n_sweeps;
  c->attempts += (uint64_t)n_sweeps * (uint64_t)c->plan.n;
  return HB_OK;
}

bool fused_kernel(const hb_ctx* c) {
  return (c->plan.engine == ENGINE_SC && c->sc_kernel == 2) || (c->plan.engine == ENGINE_BRAVAIS && c->br_kernel == 2);
}

// one sweep; with dev_out != nullptr (and fused_blocks() > 0) the colour passes also reduce M and E of
// the state they leave behind, and dev_out receives (sum Sx, sum Sy, sum Sz, E).  counted: the accepted moves of the
// sweep are added to the device counter behind hb_stats (in the measuring passes, else through the diagnostic variant)
int one_sweep(hb_ctx* c, float beta, Diag d, double* dev_out = nullptr, bool counted = false) {
  const SweepParams p = params(c, beta);
  const int fb = dev_out ? fused_blocks(c) : 0;
  if (fused_kernel(c) && !d.accept && !d.n_accept && (fb || !counted)) return fused_sweeps_launch(c, beta, 1, fb ? dev_out : nullptr, counted);
  if (counted && !fb) d.n_accept = c->counters();
  if (counted || d.n_accept) c->stat_attempts += (uint64_t)c->plan.n;
  for (int colour = 0; colour < c->n_colours; ++colour) {
    Meas m{nullptr, 0, nullptr};
    // sc: the last colour carries the whole exchange energy; bcc/fcc: every colour charges its bonds to lower colours
    if (fb) m = Meas{c->partials() + (size_t)colour * fb * 4,
                     (c->plan.engine == ENGINE_BRAVAIS || colour == c->n_colours - 1) ? 2 : 1, (counted && !d.n_accept) ? c->counters() : nullptr};
    const int rc = one_colour(c, colour, p, d, m);
    if (rc != HB_OK) return rc;
  }
  if (fb) {
    HB_CUDA(c, launch_reduce_final(c->stream, c->partials(), c->n_colours * fb, dev_out));
    c->launches += 1;
  }
  c->sweep += 1;
  c->attempts += (uint64_t)c->plan.n;
  return HB_OK;
}

// ---- replayed launches ---------------------------------------------------------------------
// Lattices whose colour pass is shorter than the gap between two kernel launches (c1, c2, most of c3 and c5) are
// bound by the launch rate.  hb_sweep then replays a CUDA graph of kGraphSweeps sweeps; the Philox sweep counter of
// a replayed launch is a device counter plus the sweep's index inside the graph (SweepParams::sweep_dev).
constexpr int kGraphSweeps = 8;

bool graph_wanted(const hb_ctx* c) {
  if (c->graph_mode == 0 || coop_mode(c) != 0 || fused_kernel(c)) return false;   // fused launches carry whole sweeps already
  return c->graph_mode == 1 || c->plan.n <= (int64_t(1) << 23);
}

int build_graph(hb_ctx* c, float beta, int meas) {
  if (c->gexec[meas]) { cudaGraphExecDestroy(c->gexec[meas]); c->gexec[meas] = nullptr; }
  if (!c->cap_stream) HB_CUDA(c, cudaStreamCreateWithFlags(&c->cap_stream, cudaStreamNonBlocking));
  cudaStream_t user = c->stream;
  const uint64_t launches = c->launches;
  const int fb = meas ? fused_blocks(c) : 0;
  HB_CUDA(c, cudaStreamBeginCapture(c->cap_stream, cudaStreamCaptureModeThreadLocal));
  c->stream = c->cap_stream;            // the launch helpers enqueue on the context's stream
  int rc = HB_OK;
  cudaError_t e = cudaSuccess;
  SweepParams p = params(c, beta);
  p.sweep_dev = c->sweep_dev();
  p.sweep_hi = 0;
  for (int u = 0; u < kGraphSweeps && rc == HB_OK && e == cudaSuccess; ++u) {
    p.sweep_lo = (uint32_t)u;
    for (int colour = 0; colour < c->n_colours && rc == HB_OK; ++colour) {
      Meas m{nullptr, 0, nullptr};
      if (fb) m = Meas{c->partials() + (size_t)colour * fb * 4,
                       (c->plan.engine == ENGINE_BRAVAIS || colour == c->n_colours - 1) ? 2 : 1, c->counters()};
      rc = one_colour(c, colour, p, Diag{nullptr, nullptr}, m);
    }
    if (fb && rc == HB_OK)
      e = launch_reduce_final_series(c->cap_stream, c->partials(), c->n_colours * fb, c->series(), c->series_idx());
  }
  if (rc == HB_OK && e == cudaSuccess) e = launch_set_counter(c->cap_stream, c->sweep_dev(), kGraphSweeps, true);
  c->stream = user;
  c->launches = launches;
  cudaGraph_t g = nullptr;
  const cudaError_t e2 = cudaStreamEndCapture(c->cap_stream, &g);
  if (rc != HB_OK) { if (g) cudaGraphDestroy(g); return rc; }
  if (e == cudaSuccess) e = e2;
  if (e == cudaSuccess) e = cudaGraphInstantiate(&c->gexec[meas], g, 0);
  if (g) cudaGraphDestroy(g);
  if (e != cudaSuccess) { c->gexec[meas] = nullptr; return fail(c, HB_ECUDA, std::string("graph capture: ") + cudaGetErrorString(e)); }
  c->g_beta[meas] = beta;
  c->g_dirty[meas] = false;
  return HB_OK;
}

// `replays` whole graphs: plain sweeps (meas = 0), or sweeps whose measurements fill the series buffer from entry 0
int graph_sweeps(hb_ctx* c, float beta, int64_t replays, int meas) {
  if (replays < 1) return HB_OK;
  if (!c->gexec[meas] || c->g_dirty[meas] || c->g_beta[meas] != beta) {
    const int rc = build_graph(c, beta, meas);
    if (rc != HB_OK) return rc;
  }
  HB_CUDA(c, launch_set_counter(c->stream, c->sweep_dev(), c->sweep, false));
  if (meas) HB_CUDA(c, launch_set_counter(c->stream, c->series_idx(), 0, false));
  for (int64_t r = 0; r < replays; ++r) HB_CUDA(c, cudaGraphLaunch(c->gexec[meas], c->stream));
  const int64_t m = replays * kGraphSweeps;
  c->launches += 1 + (meas ? 1 : 0) + (uint64_t)replays * ((uint64_t)kGraphSweeps * (c->n_colours + (meas ? 1 : 0)) + 1);
  c->sweep += (uint64_t)m;
  c->attempts += (uint64_t)m * (uint64_t)c->plan.n;
  if (meas) c->stat_attempts += (uint64_t)m * (uint64_t)c->plan.n;
  return HB_OK;
}

// ---- replicas (plan.R > 1): every replica in one thread block of one launch ------------------------------------
void select_replica(hb_ctx* c, int32_t r) {
  c->sel = r;
  c->spins = c->spins_base + (size_t)r * 3 * (size_t)c->plan.n;
  c->seed = c->seed_base + (uint64_t)r;
}

// n sweeps of all replicas at the temperatures beta[0..R) (host); series (device, R x kSeriesChunk x 4) or nullptr
int replica_sweeps(hb_ctx* c, const float* beta, int64_t n_sweeps, double* series) {
  HB_CUDA(c, cudaMemcpyAsync(c->betas(), beta, (size_t)c->plan.R * sizeof(float), cudaMemcpyHostToDevice, c->stream));
  SweepParams p = params(c, beta[0]);
  p.seed_lo = (uint32_t)c->seed_base; p.seed_hi = (uint32_t)(c->seed_base >> 32);
  const int64_t chunk = series ? kSeriesChunk : (int64_t(1) << 20);
  for (int64_t s0 = 0; s0 < n_sweeps; s0 += chunk) {
    const int m = (int)(n_sweeps - s0 < chunk ? n_sweeps - s0 : chunk);
    HB_CUDA(c, launch_sweeps_sc_coop(c->stream, c->spins_base, c->sc, c->tile, p, c->sweep, m, true, c->partials_each(), series,
                                     series ? nullptr : c->cached_each(), c->plan.R, c->betas(), (uint64_t)kSeriesChunk * 4, c->counters()));
    c->stat_attempts += (uint64_t)(series ? m : 1) * (uint64_t)c->plan.n * (uint64_t)c->plan.R;
    c->launches += 1;
    c->sweep += (uint64_t)m;
    c->attempts += (uint64_t)m * (uint64_t)c->plan.n * (uint64_t)c->plan.R;
    if (series) break;   // the caller copies a chunk out before the next one
  }
  return HB_OK;
}

int measure_into(hb_ctx* c, double* dev_out) {
  const SweepParams p = params(c, 0.0f);
  if (c->plan.engine == ENGINE_SC)
    HB_CUDA(c, launch_measure_sc(c->stream, c->spins, c->sc, c->tile.V, p, c->partials(), dev_out));
  else if (c->plan.engine == ENGINE_BRAVAIS)
    HB_CUDA(c, launch_measure_bravais(c->stream, c->spins, c->br, c->tile.V, p, c->partials(), dev_out));
  else if (c->plan.ell)
    HB_CUDA(c, launch_measure_ell(c->stream, c->spins, c->ell, p, c->partials(), dev_out));
  else
    HB_CUDA(c, launch_measure_csr(c->stream, c->spins, c->csr, p, c->partials(), dev_out));
  c->launches += 2;
  return HB_OK;
}

int check_T(hb_ctx* c, float T, float* beta) {
  if (!(T > 0.0f)) return fail(c, HB_EINVAL, "temperature must be > 0 (NaN and T <= 0 are rejected)");
  *beta = 1.0f / T;   // computed once on the host, passed to every kernel
  return HB_OK;
}

}  // namespace

// include/hb.h promises that nothing throws across the C ABI, but the host side builds tables in std::vector / std::string
// (a c5-size neighbour table is hundreds of megabytes): every entry point is a function-try-block that ends in HB_CATCH,
// so that a failed host allocation comes back as HB_ENOMEM instead of std::terminate.  A context handed out by hb_create
// before the exception stays valid for hb_error_detail / hb_destroy.
#define HB_CATCH catch (const std::bad_alloc&) { return HB_ENOMEM; } catch (const std::length_error&) { return HB_ENOMEM; } catch (...) { return HB_EINVAL; }
extern "C" {

int hb_sizes(const hb_lattice* lat, int64_t* n_sites, size_t* spins_bytes, size_t* workspace_bytes) try {
  Plan p;
  std::string why;
  if (!lat) return HB_EINVAL;
  hb_lattice padded;
  int rc = pad_slab(lat, padded, why);
  if (rc != HB_OK) return rc;
  rc = make_plan(&padded, p, why);
  if (rc != HB_OK) return rc;
  if (n_sites) *n_sites = lat->slab_Lz > 0 ? (int64_t)lat->Lx * lat->Ly * lat->Lz * (lat->kind == HB_SC ? 1 : (lat->kind == HB_BCC ? 2 : 4)) : p.n;   // a slab's own sites
  if (lat->slab_Lz > 0) p.spins_bytes += kAlign;   // the neighbour flags live behind the spins, where a peer mapping of the buffer reaches them
  if (spins_bytes) *spins_bytes = p.spins_bytes;
  if (workspace_bytes) *workspace_bytes = p.ws_bytes;
  return HB_OK;
} HB_CATCH

int hb_create(hb_ctx** out, const hb_lattice* lat, float J, float K, const float e[3], uint64_t seed,
              const hb_buffers* bufs) try {
  if (!out) return HB_EINVAL;
  *out = nullptr;
  hb_ctx* c = new (std::nothrow) hb_ctx;
  if (!c) return HB_ENOMEM;
  // the context is handed back even on failure so that hb_error_detail can say why
  *out = c;
  std::string why;
  if (!lat) { c->sticky = HB_EINVAL; return fail(c, HB_EINVAL, "lattice is NULL"); }
  hb_lattice padded;
  int rc = pad_slab(lat, padded, why);
  if (rc != HB_OK) { c->sticky = rc; return fail(c, rc, why); }
  if (lat->slab_Lz > 0) { c->slab_Lz = lat->slab_Lz; c->slab_z0 = lat->slab_z0; }
  lat = &padded;
  rc = make_plan(lat, c->plan, why);
  if (rc != HB_OK) { c->sticky = rc; return fail(c, rc, why); }
  if (c->slab_Lz > 0) c->plan.spins_bytes += kAlign;   // neighbour flags behind the spins (hb_sizes)
  if (!e || !unit_vector(e) || !std::isfinite(J) || !std::isfinite(K)) {
    c->sticky = HB_EINVAL;
    return fail(c, HB_EINVAL, "J, K must be finite and e a unit vector");
  }
  c->kind = lat->kind; c->Lx = lat->Lx; c->Ly = lat->Ly; c->Lz = lat->Lz;
  c->J = J; c->K = K; c->e[0] = e[0]; c->e[1] = e[1]; c->e[2] = e[2];
  c->seed = c->seed_base = seed;
  const Plan& P = c->plan;
  if (P.per_site)
    for (int64_t i = 0; i < P.n; ++i)
      if (!unit_vector(lat->e_site + 3 * i) || !std::isfinite(lat->K_site[i])) {
        c->sticky = HB_EINVAL;
        return fail(c, HB_EINVAL, "e_site must hold unit vectors and K_site finite values");
      }

  // ---- host tables -------------------------------------------------------------------------
  HostCsr g;
  const int64_t* row_ptr = nullptr;
  const int32_t* col = nullptr;
  if (P.engine == ENGINE_CSR) {
    if (lat->kind == HB_CSR) {
      const int64_t n_own = P.part_total > 0 ? P.n_own : P.n;
      why = validate_csr(P.n, lat->row_ptr, lat->col_idx, n_own);
      if (!why.empty()) { c->sticky = HB_EINVAL; return fail(c, HB_EINVAL, why); }
      row_ptr = lat->row_ptr; col = lat->col_idx;
      if (lat->colour) {
        why = validate_colouring(P.n, row_ptr, col, lat->colour, lat->n_colours, n_own);
        if (!why.empty()) { c->sticky = HB_EINVAL; return fail(c, HB_EINVAL, why); }
        c->colour_host.assign(lat->colour, lat->colour + P.n);
        c->n_colours = lat->n_colours;
      } else {
        g.n = P.n;
        g.row_ptr.assign(row_ptr, row_ptr + P.n + 1);
        g.col.assign(col, col + P.nnz);
        greedy_first_fit(g);
        c->colour_host = g.colour;
        c->n_colours = g.n_colours;
      }
    } else {
      if (lat->kind == HB_BCC) build_bcc_csr(lat->Lx, lat->Ly, lat->Lz, g);
      else if (lat->kind == HB_FCC) build_fcc_csr(lat->Lx, lat->Ly, lat->Lz, g);
      else {  // sc with per-site anisotropy: explicit table, same order -x,+x,-y,+y,-z,+z
        const int32_t Lx = lat->Lx, Ly = lat->Ly, Lz = lat->Lz;
        g.n = P.n; g.n_colours = 2;
        g.row_ptr.resize(P.n + 1); g.col.resize(6 * P.n); g.colour.resize(P.n);
        for (int64_t i = 0; i <= P.n; ++i) g.row_ptr[i] = 6 * i;
        for (int32_t z = 0; z < Lz; ++z)
          for (int32_t y = 0; y < Ly; ++y)
            for (int32_t x = 0; x < Lx; ++x) {
              const int64_t plane = (int64_t)z * Ly, i = (plane + y) * Lx + x;
              int32_t* o = &g.col[6 * i];
              o[0] = (int32_t)((plane + y) * Lx + (x ? x - 1 : Lx - 1));
              o[1] = (int32_t)((plane + y) * Lx + (x + 1 < Lx ? x + 1 : 0));
              o[2] = (int32_t)((plane + (y ? y - 1 : Ly - 1)) * Lx + x);
              o[3] = (int32_t)((plane + (y + 1 < Ly ? y + 1 : 0)) * Lx + x);
              o[4] = (int32_t)(((int64_t)(z ? z - 1 : Lz - 1) * Ly + y) * Lx + x);
              o[5] = (int32_t)(((int64_t)(z + 1 < Lz ? z + 1 : 0) * Ly + y) * Lx + x);
              g.colour[i] = (x + y + z) & 1;
            }
      }
      row_ptr = g.row_ptr.data(); col = g.col.data();
      c->colour_host = g.colour;
      c->n_colours = g.n_colours;
    }
  } else if (P.engine == ENGINE_BRAVAIS) {
    c->n_colours = lat->kind == HB_BCC ? 2 : 4;       // colour = basis index
    c->br.kind = lat->kind; c->br.Lx = lat->Lx; c->br.Ly = lat->Ly; c->br.Lz = lat->Lz;
    c->br.n = (uint32_t)P.n; c->br.nc = (uint32_t)(P.n / c->n_colours);
    c->br.ghost = 0; c->br.nc_id = c->br.nc; c->br.cell_base = 0;
    if (c->slab_Lz > 0) {   // local cell plane 1 is global plane slab_z0 (lat is the padded description here: Lz + 2 planes)
      c->br.ghost = 1;
      c->br.nc_id = (uint32_t)((int64_t)lat->Lx * lat->Ly * c->slab_Lz);
      c->br.cell_base = (uint32_t)(((int64_t)c->slab_z0 - 1) * lat->Ly * lat->Lx);
      c->graph_mode = 0; c->fused_measure = false;
    }
    c->tile = default_tile(lat->Lx, lat->Ly, lat->Lz);
    // The warp-specialised kernel pays on lattices far larger than L2: bcc +2 ... +10 % over the direct kernel
    // (33.5 M sites, rows of 64 / 128 / 256 cells: 112 / 117 / 125 against 109 / 108 / 114 Gupd/s); fcc only with all passes in one
    // launch and long rows (89.9 against 85.1), its staged groups being three sublattices wide.  c2 and c3 (0.5 M and 8.4 M
    // sites, L2-resident, a handful of plane steps per CTA and pass) stay on the direct kernel: 27 against 70, 59 against 80.
    if (bravais_ws_supported(c->br) && P.n >= (int64_t(1) << 24)) {   // (never a slab: bravais_ws_supported)
      if (lat->kind == HB_BCC) { c->br_kernel = 1; c->br_zt = (lat->Lx > 64 && lat->Lx <= 128) ? 8 : 16; }
      else if (lat->Lx > 128) { c->br_kernel = 2; c->br_zt = 16; }
      if (c->br_zt > lat->Lz) c->br_zt = lat->Lz;
    }
    {
      int dev = 0, sms = 0;
      if (cudaGetDevice(&dev) == cudaSuccess && cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && sms > 0)
        c->n_sms = sms;
      cudaGetLastError();
    }
    clamp_bravais_ws(c);   // (needs n_sms: the chunk count depends on the grid)
  } else {
    c->n_colours = 2;
    c->sc.Lx = lat->Lx; c->sc.Ly = lat->Ly; c->sc.Lz = lat->Lz;
    c->sc.H = lat->Lx / 2; c->sc.n = (uint32_t)P.n; c->sc.half = (uint32_t)(P.n / 2);
    c->tile = default_tile(c->sc.H, c->sc.Ly, c->sc.Lz);
    {
      int dev = 0, sms = 0;
      if (cudaGetDevice(&dev) == cudaSuccess && cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && sms > 0)
        c->n_sms = sms;
      cudaGetLastError();
    }
    if (c->ws_zt > c->sc.Lz) c->ws_zt = c->sc.Lz;
    // the warp-specialised kernel is built for long rows (pitch 1024 B): with them, on lattices far larger than L2, it
    // sustains 3-4 % more than the direct kernel and stays below the power cap; everything else runs direct
    c->sc_kernel = (sc_ws_supported(c->sc) && (c->sc.H >= 224 || (c->sc.H >= 112 && c->sc.H <= 128)) && P.n >= (int64_t(1) << 24)) ? 1 : 0;
    if (c->slab_Lz > 0) {   // local plane 1 is global plane slab_z0; graphs, persistent kernels and the fused measurement are for whole lattices
      c->sc.ghost = 1;
      c->sc.site_base = (uint32_t)(((int64_t)c->slab_z0 - 1) * lat->Ly * lat->Lx);
      c->graph_mode = 0; c->sc_coop = 0; c->fused_measure = false;
    }
    if (c->sc.H <= 128) c->ws_variant = 5;   // rows of 112-128 floats (256^3): 8-row tiles at a 512-byte pitch, +2.5 % over the direct kernel
    else c->ws_variant = sc_ws_variant_supported(c->sc, 4) ? 4 : 2;   // 7-row tiles where the rows fit them (c4: +2 %), else 4-row tiles
  }

  // programmatic stream serialisation of the colour launches: mode 1 (the next launch comes in as blocks
  // exit) was measured to pay on every engine and size; mode 2 crowds the single wave of small launches
  c->pdl = 1;
  if (P.ell) c->csr_block = 64;   // ELL kernel: blocks of 64 threads (c5 greedy colouring 29.2 against 28.5 Gupd/s with 128)

  // ---- device memory --------------------------------------------------------------------------
  if (bufs) {
    if (!bufs->spins || !bufs->workspace || bufs->spins_bytes < P.spins_bytes || bufs->workspace_bytes < P.ws_bytes ||
        ((uintptr_t)bufs->spins % kAlign) || ((uintptr_t)bufs->workspace % kAlign)) {
      c->sticky = HB_ENOMEM;
      return fail(c, HB_ENOMEM, "caller buffers are NULL, too small (see hb_sizes) or not 256-byte aligned");
    }
    c->spins = c->spins_base = static_cast<float*>(bufs->spins);
    c->ws = static_cast<char*>(bufs->workspace);
    c->stream = static_cast<cudaStream_t>(bufs->cuda_stream);
  } else {
    void* a = nullptr; void* b = nullptr;
    if (cudaMalloc(&a, P.spins_bytes) != cudaSuccess || cudaMalloc(&b, P.ws_bytes) != cudaSuccess) {
      if (a) cudaFree(a);
      cudaGetLastError();
      c->sticky = HB_ENOMEM;
      return fail(c, HB_ENOMEM, "cudaMalloc failed");
    }
    c->spins = c->spins_base = static_cast<float*>(a); c->ws = static_cast<char*>(b);
    c->own_spins = c->own_ws = true;
  }
  HB_CUDA(c, cudaMemsetAsync(c->ws + P.off_counters, 0, kAlign, c->stream));
  if (c->slab_Lz > 0) HB_CUDA(c, cudaMemsetAsync(c->slab_flags(), 0, kAlign, c->stream));
  if (P.engine == ENGINE_SC || P.engine == ENGINE_BRAVAIS) HB_CUDA(c, cudaMemsetAsync(c->ws + P.off_wsdone, 0, (size_t)kWsDoneWords * sizeof(uint32_t), c->stream));

  if (P.engine == ENGINE_CSR) {
    // sites sorted by (colour, id): one contiguous list segment per colour; the ghost sites of a part follow the last colour
    const int64_t n_own = P.part_total > 0 ? P.n_own : P.n;
    std::vector<uint32_t> count((size_t)c->n_colours + 1, 0);
    for (int64_t i = 0; i < n_own; ++i) count[c->colour_host[i] + 1] += 1;
    for (int k = 0; k < c->n_colours; ++k) count[k + 1] += count[k];
    c->colour_begin = count;
    if (c->n_colours > kMaxColours) { c->sticky = HB_EINVAL; return fail(c, HB_EINVAL, "more than 65536 colours"); }
    std::vector<int32_t> list((size_t)P.n);
    {
      std::vector<uint32_t> cur(count.begin(), count.end() - 1);
      for (int64_t i = 0; i < n_own; ++i) list[cur[c->colour_host[i]]++] = (int32_t)i;
      for (int64_t i = n_own; i < P.n; ++i) list[i] = (int32_t)i;
    }
    int32_t* d_list = reinterpret_cast<int32_t*>(c->ws + P.off_list);
    HB_CUDA(c, cudaMemcpyAsync(d_list, list.data(), list.size() * 4, cudaMemcpyHostToDevice, c->stream));
    std::vector<int32_t> rp32, ell, inv;
    std::vector<float> soa;
    if (P.ell) {
      // internal order m = position in the colour-sorted list; table entries are internal indices
      inv.resize((size_t)P.n);
      for (int64_t m = 0; m < P.n; ++m) inv[list[m]] = (int32_t)m;
      ell.assign((size_t)P.maxdeg * (size_t)P.n, -1);
      for (int k = 0; k < c->n_colours; ++k) {
        const size_t begin = count[k], nc = count[k + 1] - count[k];
        for (size_t t = 0; t < nc; ++t) {
          const int64_t id = list[begin + t];
          int32_t* e0 = ell.data() + (size_t)P.maxdeg * begin + t;
          for (int64_t q = row_ptr[id]; q < row_ptr[id + 1]; ++q) e0[(size_t)(q - row_ptr[id]) * nc] = inv[col[q]];
        }
      }
      int32_t* d_ell = reinterpret_cast<int32_t*>(c->ws + P.off_ell);
      uint32_t* d_cb = reinterpret_cast<uint32_t*>(c->ws + P.off_cbegin);
      HB_CUDA(c, cudaMemcpyAsync(d_ell, ell.data(), ell.size() * 4, cudaMemcpyHostToDevice, c->stream));
      HB_CUDA(c, cudaMemcpyAsync(d_cb, count.data(), count.size() * 4, cudaMemcpyHostToDevice, c->stream));
      c->ell.n = (uint32_t)P.n; c->ell.maxdeg = (uint32_t)P.maxdeg; c->ell.ell = d_ell; c->ell.perm = d_list;
      c->ell.colour_begin = d_cb; c->ell.n_colours = c->n_colours;
      c->ell.site_base = (uint32_t)P.part_first; c->ell.inv = nullptr;
      if (P.part_total > 0) {
        int32_t* d_inv = reinterpret_cast<int32_t*>(c->ws + P.off_inv);
        HB_CUDA(c, cudaMemcpyAsync(d_inv, inv.data(), inv.size() * 4, cudaMemcpyHostToDevice, c->stream));
        c->ell.inv = d_inv;
      }
      c->ell.K = c->ell.ex = c->ell.ey = c->ell.ez = nullptr;
      if (P.per_site) {   // (K, e) in internal order, one plane each: K at off_K, ex|ey|ez at off_e
        soa.resize(4 * (size_t)P.n);
        for (int64_t m = 0; m < P.n; ++m) {
          const int64_t id = list[m];
          soa[m] = lat->K_site[id];
          soa[(size_t)P.n + m] = lat->e_site[3 * id];
          soa[2 * (size_t)P.n + m] = lat->e_site[3 * id + 1];
          soa[3 * (size_t)P.n + m] = lat->e_site[3 * id + 2];
        }
        float* d_K = reinterpret_cast<float*>(c->ws + P.off_K);
        float* d_e = reinterpret_cast<float*>(c->ws + P.off_e);
        HB_CUDA(c, cudaMemcpyAsync(d_K, soa.data(), (size_t)P.n * 4, cudaMemcpyHostToDevice, c->stream));
        HB_CUDA(c, cudaMemcpyAsync(d_e, soa.data() + P.n, (size_t)P.n * 12, cudaMemcpyHostToDevice, c->stream));
        c->ell.K = d_K; c->ell.ex = d_e; c->ell.ey = d_e + P.n; c->ell.ez = d_e + 2 * (size_t)P.n;
      }
    } else {
      rp32.resize((size_t)P.n + 1);
      for (int64_t i = 0; i <= P.n; ++i) rp32[i] = (int32_t)row_ptr[i];
      int32_t* d_rp = reinterpret_cast<int32_t*>(c->ws + P.off_row_ptr);
      int32_t* d_col = reinterpret_cast<int32_t*>(c->ws + P.off_col);
      HB_CUDA(c, cudaMemcpyAsync(d_rp, rp32.data(), rp32.size() * 4, cudaMemcpyHostToDevice, c->stream));
      if (P.nnz) HB_CUDA(c, cudaMemcpyAsync(d_col, col, (size_t)P.nnz * 4, cudaMemcpyHostToDevice, c->stream));
      c->csr.n = (uint32_t)P.n; c->csr.row_ptr = d_rp; c->csr.col = d_col; c->csr.list = d_list;
      c->csr.n_own = (uint32_t)n_own; c->csr.site_base = (uint32_t)P.part_first;
      c->csr.K_site = nullptr; c->csr.e_site = nullptr;
      if (P.per_site) {
        float* d_K = reinterpret_cast<float*>(c->ws + P.off_K);
        float* d_e = reinterpret_cast<float*>(c->ws + P.off_e);
        HB_CUDA(c, cudaMemcpyAsync(d_K, lat->K_site, (size_t)P.n * 4, cudaMemcpyHostToDevice, c->stream));
        HB_CUDA(c, cudaMemcpyAsync(d_e, lat->e_site, (size_t)P.n * 12, cudaMemcpyHostToDevice, c->stream));
        c->csr.K_site = d_K; c->csr.e_site = d_e;
      }
    }
    HB_CUDA(c, cudaStreamSynchronize(c->stream));   // the host vectors die at return
  }
  return HB_OK;
} HB_CATCH

int hb_destroy(hb_ctx* c) try {
  if (!c) return HB_OK;
  for (int k = 0; k < 2; ++k) if (c->gexec[k]) cudaGraphExecDestroy(c->gexec[k]);
  if (c->cap_stream) cudaStreamDestroy(c->cap_stream);
  if (c->stage_stream) { cudaStreamSynchronize(c->stage_stream); cudaStreamDestroy(c->stage_stream); }
  if (c->stage_filled) cudaEventDestroy(c->stage_filled);
  if (c->stage_free) cudaEventDestroy(c->stage_free);
  if (c->stage) cudaFree(c->stage);
  if (c->own_spins && c->spins_base) cudaFree(c->spins_base);
  if (c->own_ws && c->ws) cudaFree(c->ws);
  delete c;
  return HB_OK;
} HB_CATCH

int hb_init_random(hb_ctx* c) try {
  HB_CHECK_CTX(c);
  c->cache_valid = false;
  c->each_valid = false;
  if (c->plan.R > 1) {
    for (int32_t r = 0; r < c->plan.R; ++r) {
      const uint64_t sd = c->seed_base + (uint64_t)r;
      HB_CUDA(c, launch_init_random_sc(c->stream, c->spins_base + (size_t)r * 3 * (size_t)c->plan.n, c->sc, (uint32_t)sd, (uint32_t)(sd >> 32)));
    }
    c->launches += (uint64_t)c->plan.R;
    c->initialised = true;
    return HB_OK;
  }
  if (c->plan.engine == ENGINE_SC)
    HB_CUDA(c, launch_init_random_sc(c->stream, c->spins, c->sc, (uint32_t)c->seed, (uint32_t)(c->seed >> 32)));
  else if (c->plan.ell)
    HB_CUDA(c, launch_init_random_perm(c->stream, c->spins, c->ell.perm, (uint32_t)c->plan.n, (uint32_t)c->seed, (uint32_t)(c->seed >> 32), c->ell.site_base));
  else if (c->plan.engine == ENGINE_BRAVAIS)
    HB_CUDA(c, launch_init_random_bravais(c->stream, c->spins, c->br, (uint32_t)c->seed, (uint32_t)(c->seed >> 32)));
  else
    HB_CUDA(c, launch_init_random_flat(c->stream, c->spins, (uint32_t)c->plan.n, (uint32_t)c->seed, (uint32_t)(c->seed >> 32), (uint32_t)c->plan.part_first));
  c->launches += 1;
  c->initialised = true;
  return HB_OK;
} HB_CATCH

int hb_init_aligned(hb_ctx* c, const float dir[3]) try {
  HB_CHECK_CTX(c);
  if (!dir || !unit_vector(dir)) return fail(c, HB_EINVAL, "dir must be a unit vector");
  c->cache_valid = false;
  c->each_valid = false;
  if (c->plan.R > 1) {
    for (int32_t r = 0; r < c->plan.R; ++r)
      HB_CUDA(c, launch_fill(c->stream, c->spins_base + (size_t)r * 3 * (size_t)c->plan.n, (uint32_t)c->plan.n, dir[0], dir[1], dir[2]));
    c->launches += (uint64_t)c->plan.R;
    c->initialised = true;
    return HB_OK;
  }
  if (c->plan.ell) HB_CUDA(c, launch_fill_ell(c->stream, c->spins, (uint32_t)c->plan.n, dir[0], dir[1], dir[2]));
  else HB_CUDA(c, launch_fill(c->stream, c->spins, (uint32_t)c->plan.n, dir[0], dir[1], dir[2]));
  c->launches += 1;
  c->initialised = true;
  return HB_OK;
} HB_CATCH

int hb_set_spins(hb_ctx* c, const float* sx, const float* sy, const float* sz) try {
  HB_CHECK_CTX(c);
  c->cache_valid = false;
  if (!sx || !sy || !sz) return fail(c, HB_EINVAL, "NULL spin array");
  c->each_valid = false;
  const size_t n = (size_t)c->plan.n;
  // slab: the caller's Lx Ly Lz sites sit between two ghost planes (zero until exchanged): they are copied into the middle
  // of the zeroed staging plane, no padded host copy is made
  const size_t skip = (c->slab_Lz > 0 && c->plan.engine == ENGINE_SC) ? (size_t)c->sc.Lx * c->sc.Ly : 0;
  const float* src[3] = {sx, sy, sz};
  for (int k = 0; k < 3; ++k) {
    if (c->plan.engine == ENGINE_BRAVAIS && c->slab_Lz > 0) {
      // a bcc / fcc slab: the own cell planes of every sublattice are one contiguous run between its two ghost planes
      const size_t plane = (size_t)c->br.Lx * c->br.Ly, own = (size_t)c->br.nc - 2 * plane;
      HB_CUDA(c, cudaMemsetAsync(c->spins + k * n, 0, n * 4, c->stream));
      for (int b = 0; b < c->n_colours; ++b)
        HB_CUDA(c, cudaMemcpyAsync(c->spins + k * n + (size_t)b * c->br.nc + plane, src[k] + (size_t)b * own, own * 4, cudaMemcpyHostToDevice, c->stream));
    } else if (c->plan.engine == ENGINE_SC) {
      if (skip) HB_CUDA(c, cudaMemsetAsync(c->staging(), 0, n * 4, c->stream));
      HB_CUDA(c, cudaMemcpyAsync(c->staging() + skip, src[k], (n - 2 * skip) * 4, cudaMemcpyHostToDevice, c->stream));
      HB_CUDA(c, launch_sc_permute(c->stream, c->spins + k * n, c->staging(), c->sc, true));
      c->launches += 1;
    } else if (c->plan.ell) {
      HB_CUDA(c, cudaMemcpyAsync(c->staging(), src[k], n * 4, cudaMemcpyHostToDevice, c->stream));
      HB_CUDA(c, launch_permute_ell(c->stream, c->spins, c->staging(), c->ell.perm, (uint32_t)n, k, true));
      c->launches += 1;
    } else {
      HB_CUDA(c, cudaMemcpyAsync(c->spins + k * n, src[k], n * 4, cudaMemcpyHostToDevice, c->stream));
    }
  }
  HB_CUDA(c, cudaStreamSynchronize(c->stream));   // the caller may reuse its arrays
  c->initialised = true;
  return HB_OK;
} HB_CATCH

// ---- staged upload: the host->device copy of the NEXT state overlaps the sweeps of the current one ---------------------------
int hb_stage_spins(hb_ctx* c, const float* sx, const float* sy, const float* sz) try {
  HB_CHECK_CTX(c);
  if (!sx || !sy || !sz) return fail(c, HB_EINVAL, "NULL spin array");
  if (c->slab_Lz > 0 || c->plan.part_total > 0 || c->plan.R > 1) return fail(c, HB_EINVAL, "hb_stage_spins: whole lattices without replicas");
  // a second upload would overwrite the area while the first may still be in flight from host arrays the caller no longer holds
  if (c->stage_pending) return fail(c, HB_ESTATE, "hb_stage_spins: a staged state is waiting for hb_commit_spins");
  const size_t n = (size_t)c->plan.n;
  if (!c->stage) {
    if (cudaMalloc(reinterpret_cast<void**>(&c->stage), 3 * n * sizeof(float)) != cudaSuccess) { cudaGetLastError(); return fail(c, HB_ENOMEM, "hb_stage_spins: cudaMalloc of the upload area failed"); }
    HB_CUDA(c, cudaStreamCreateWithFlags(&c->stage_stream, cudaStreamNonBlocking));
    HB_CUDA(c, cudaEventCreateWithFlags(&c->stage_filled, cudaEventDisableTiming));
    HB_CUDA(c, cudaEventCreateWithFlags(&c->stage_free, cudaEventDisableTiming));
    HB_CUDA(c, cudaEventRecord(c->stage_free, c->stream));
  }
  HB_CUDA(c, cudaStreamWaitEvent(c->stage_stream, c->stage_free, 0));   // the last commit has read the area
  const float* src[3] = {sx, sy, sz};
  for (int k = 0; k < 3; ++k)
    HB_CUDA(c, cudaMemcpyAsync(c->stage + k * n, src[k], n * sizeof(float), cudaMemcpyHostToDevice, c->stage_stream));
  HB_CUDA(c, cudaEventRecord(c->stage_filled, c->stage_stream));
  c->stage_pending = true;
  return HB_OK;
} HB_CATCH

int hb_commit_spins(hb_ctx* c) try {
  HB_CHECK_CTX(c);
  if (!c->stage_pending) return fail(c, HB_ESTATE, "hb_commit_spins without a staged state (hb_stage_spins)");
  HB_CUDA(c, cudaEventSynchronize(c->stage_filled));                     // the caller may reuse its host arrays after this call
  c->cache_valid = c->each_valid = false;
  const size_t n = (size_t)c->plan.n;
  for (int k = 0; k < 3; ++k) {
    if (c->plan.engine == ENGINE_SC) {
      HB_CUDA(c, launch_sc_permute(c->stream, c->spins + k * n, c->stage + k * n, c->sc, true));
      c->launches += 1;
    } else if (c->plan.ell) {
      HB_CUDA(c, launch_permute_ell(c->stream, c->spins, c->stage + k * n, c->ell.perm, (uint32_t)n, k, true));
      c->launches += 1;
    } else {
      HB_CUDA(c, cudaMemcpyAsync(c->spins + k * n, c->stage + k * n, n * sizeof(float), cudaMemcpyDeviceToDevice, c->stream));
    }
  }
  HB_CUDA(c, cudaEventRecord(c->stage_free, c->stream));
  c->stage_pending = false;
  c->initialised = true;
  return HB_OK;
} HB_CATCH

int hb_get_spins(hb_ctx* c, float* sx, float* sy, float* sz) try {
  HB_CHECK_CTX(c);
  if (!sx || !sy || !sz) return fail(c, HB_EINVAL, "NULL spin array");
  if (!c->initialised) return fail(c, HB_ESTATE, "spins not initialised");
  const size_t n = (size_t)c->plan.n;
  float* dst[3] = {sx, sy, sz};
  for (int k = 0; k < 3; ++k) {
    if (c->plan.engine == ENGINE_BRAVAIS && c->slab_Lz > 0) {
      const size_t plane = (size_t)c->br.Lx * c->br.Ly, own = (size_t)c->br.nc - 2 * plane;
      for (int b = 0; b < c->n_colours; ++b)
        HB_CUDA(c, cudaMemcpyAsync(dst[k] + (size_t)b * own, c->spins + k * n + (size_t)b * c->br.nc + plane, own * 4, cudaMemcpyDeviceToHost, c->stream));
    } else if (c->plan.engine == ENGINE_SC) {
      HB_CUDA(c, launch_sc_permute(c->stream, c->staging(), c->spins + k * n, c->sc, false));
      c->launches += 1;
      // a slab hands out its own planes only: they are contiguous in canonical order, between the two ghost planes
      const size_t skip = c->slab_Lz > 0 ? (size_t)c->sc.Lx * c->sc.Ly : 0;
      HB_CUDA(c, cudaMemcpyAsync(dst[k], c->staging() + skip, (n - 2 * skip) * 4, cudaMemcpyDeviceToHost, c->stream));
    } else if (c->plan.ell) {
      HB_CUDA(c, launch_permute_ell(c->stream, c->spins, c->staging(), c->ell.perm, (uint32_t)n, k, false));
      c->launches += 1;
      HB_CUDA(c, cudaMemcpyAsync(dst[k], c->staging(), n * 4, cudaMemcpyDeviceToHost, c->stream));
    } else {
      HB_CUDA(c, cudaMemcpyAsync(dst[k], c->spins + k * n, n * 4, cudaMemcpyDeviceToHost, c->stream));
    }
  }
  HB_CUDA(c, cudaStreamSynchronize(c->stream));
  return HB_OK;
} HB_CATCH

int hb_sweep(hb_ctx* c, float T, int64_t n_sweeps) try {
  HB_CHECK_CTX(c);
  if (c->slab_Lz > 0 || c->plan.part_total > 0) return fail(c, HB_ESTATE, "slab or part context: drive it with hb_slab_pass / hb_slab_next_sweep and the exchange step (include/hb.h)");
  if (n_sweeps < 0) return fail(c, HB_EINVAL, "n_sweeps < 0");
  if (!c->initialised) return fail(c, HB_ESTATE, "spins not initialised");
  float beta;
  int rc = check_T(c, T, &beta);
  if (rc != HB_OK) return rc;
  if (n_sweeps > 0) c->cache_valid = false;
  if (c->plan.R > 1) {
    if (n_sweeps == 0) return HB_OK;
    const std::vector<float> b((size_t)c->plan.R, beta);
    c->each_valid = false;
    rc = replica_sweeps(c, b.data(), n_sweeps, nullptr);
    if (rc == HB_OK) c->each_valid = true;
    return rc;
  }
  if (n_sweeps > 0 && coop_mode(c) != 0) {
    rc = coop_sweeps(c, beta, n_sweeps, nullptr, c->cached());
    if (rc == HB_OK) c->cache_valid = true;
    return rc;
  }
  const bool fuse = fused_blocks(c) > 0;
  int64_t s = 0;
  if (graph_wanted(c)) {   // whole graphs of kGraphSweeps; the last sweep stays outside (it may carry the measurement)
    const int64_t replays = (n_sweeps - 1) / kGraphSweeps;
    rc = graph_sweeps(c, beta, replays, 0);
    if (rc != HB_OK) return rc;
    s = replays * kGraphSweeps;
  }
  if (fused_kernel(c)) {   // all but the last sweep: up to fused_sweeps sweeps per launch
    while (s < n_sweeps - 1) {
      const int g = (int)(n_sweeps - 1 - s < c->fused_sweeps ? n_sweeps - 1 - s : c->fused_sweeps);
      rc = fused_sweeps_launch(c, beta, g, nullptr, false);
      if (rc != HB_OK) return rc;
      s += g;
    }
  }
  for (; s < n_sweeps; ++s) {
    const bool last = s == n_sweeps - 1;   // carries the fused measurement and counts its accepted moves (hb_stats)
    rc = one_sweep(c, beta, Diag{nullptr, nullptr}, (fuse && last) ? c->cached() : nullptr, last);
    if (rc != HB_OK) return rc;
  }
  if (fuse && n_sweeps > 0) c->cache_valid = true;
  return HB_OK;
} HB_CATCH

int hb_measure(hb_ctx* c, double M[3], double* E) try {
  HB_CHECK_CTX(c);
  if (!M || !E) return fail(c, HB_EINVAL, "NULL output");
  if (!c->initialised) return fail(c, HB_ESTATE, "spins not initialised");
  if (c->plan.R > 1 && c->each_valid) {   // the replicas' last sweep left all measurements behind
    double h[4];
    HB_CUDA(c, cudaMemcpyAsync(h, c->cached_each() + 4 * (size_t)c->sel, sizeof h, cudaMemcpyDeviceToHost, c->stream));
    HB_CUDA(c, cudaStreamSynchronize(c->stream));
    const double inv = 1.0 / (double)c->plan.n;
    M[0] = h[0] * inv; M[1] = h[1] * inv; M[2] = h[2] * inv;
    *E = h[3];
    return HB_OK;
  }
  if (c->plan.R > 1) c->cache_valid = false;   // the single slot may hold another replica's numbers
  if (!c->cache_valid) {
    const int rc = measure_into(c, c->cached());
    if (rc != HB_OK) return rc;
    c->cache_valid = true;
  }
  double h[4];
  HB_CUDA(c, cudaMemcpyAsync(h, c->cached(), sizeof h, cudaMemcpyDeviceToHost, c->stream));
  HB_CUDA(c, cudaStreamSynchronize(c->stream));
  // a slab returns its share of M of the whole lattice (the kernel skipped the ghost planes)
  // (a part of a table likewise: its own sites over the sites of the whole table)
  const double inv = 1.0 / (c->slab_Lz > 0 ? (double)c->Lx * c->Ly * c->slab_Lz * (c->plan.engine == ENGINE_SC ? 1 : c->n_colours)
                                           : (c->plan.part_total > 0 ? (double)c->plan.part_total : (double)c->plan.n));
  M[0] = h[0] * inv; M[1] = h[1] * inv; M[2] = h[2] * inv;
  *E = h[3];
  return HB_OK;
} HB_CATCH

int hb_sweep_series(hb_ctx* c, float T, int64_t n_sweeps, double* M_series, double* E_series) try {
  HB_CHECK_CTX(c);
  if (c->slab_Lz > 0 || c->plan.part_total > 0) return fail(c, HB_ESTATE, "slab or part context: drive it with hb_slab_pass / hb_slab_next_sweep and the exchange step (include/hb.h)");
  if (n_sweeps < 0 || !M_series || !E_series) return fail(c, HB_EINVAL, "bad series arguments");
  if (c->plan.R > 1) return fail(c, HB_EINVAL, "a context with replicas takes hb_sweep_series_each");
  if (!c->initialised) return fail(c, HB_ESTATE, "spins not initialised");
  float beta;
  int rc = check_T(c, T, &beta);
  if (rc != HB_OK) return rc;
  std::vector<double> h((size_t)kSeriesChunk * 4);
  const double inv = 1.0 / (double)c->plan.n;
  const bool fuse = fused_blocks(c) > 0;
  if (n_sweeps > 0) c->cache_valid = false;
  for (int64_t s0 = 0; s0 < n_sweeps; s0 += kSeriesChunk) {
    const int64_t m = n_sweeps - s0 < kSeriesChunk ? n_sweeps - s0 : kSeriesChunk;
    if (coop_mode(c) != 0) {
      rc = coop_sweeps(c, beta, m, c->series(), nullptr);
      if (rc != HB_OK) return rc;
    } else {
    int64_t s = 0;
    if (fuse && graph_wanted(c)) {   // measured sweeps replayed: the reduction node writes entry 0, 1, 2, ... of the chunk
      const int64_t replays = m / kGraphSweeps;
      rc = graph_sweeps(c, beta, replays, 1);
      if (rc != HB_OK) return rc;
      s = replays * kGraphSweeps;
    }
    for (; s < m; ++s) {
      rc = one_sweep(c, beta, Diag{nullptr, nullptr}, fuse ? c->series() + 4 * s : nullptr, true);
      if (rc != HB_OK) return rc;
      if (!fuse) {
        rc = measure_into(c, c->series() + 4 * s);
        if (rc != HB_OK) return rc;
      }
    }
    }
    HB_CUDA(c, cudaMemcpyAsync(h.data(), c->series(), (size_t)m * 32, cudaMemcpyDeviceToHost, c->stream));
    HB_CUDA(c, cudaStreamSynchronize(c->stream));
    for (int64_t s = 0; s < m; ++s) {
      M_series[3 * (s0 + s) + 0] = h[4 * s + 0] * inv;
      M_series[3 * (s0 + s) + 1] = h[4 * s + 1] * inv;
      M_series[3 * (s0 + s) + 2] = h[4 * s + 2] * inv;
      E_series[s0 + s] = h[4 * s + 3];
    }
  }
  return HB_OK;
} HB_CATCH

int hb_sweep_record(hb_ctx* c, float T, uint8_t* accept) try {
  HB_CHECK_CTX(c);
  if (c->slab_Lz > 0 || c->plan.part_total > 0) return fail(c, HB_ESTATE, "slab or part context: drive it with hb_slab_pass / hb_slab_next_sweep and the exchange step (include/hb.h)");
  if (!accept) return fail(c, HB_EINVAL, "NULL accept array");
  if (c->plan.R > 1) return fail(c, HB_EINVAL, "hb_sweep_record needs a context without replicas");
  if (!c->initialised) return fail(c, HB_ESTATE, "spins not initialised");
  float beta;
  int rc = check_T(c, T, &beta);
  if (rc != HB_OK) return rc;
  uint8_t* d_acc = reinterpret_cast<uint8_t*>(c->staging());
  HB_CUDA(c, cudaMemsetAsync(d_acc, 0xFF, (size_t)c->plan.n, c->stream));   // every site must be overwritten
  c->cache_valid = false;
  rc = one_sweep(c, beta, Diag{d_acc, c->counters()});
  if (rc != HB_OK) return rc;
  HB_CUDA(c, cudaMemcpyAsync(accept, d_acc, (size_t)c->plan.n, cudaMemcpyDeviceToHost, c->stream));
  HB_CUDA(c, cudaStreamSynchronize(c->stream));
  return HB_OK;
} HB_CATCH

int hb_select_replica(hb_ctx* c, int32_t replica) try {
  HB_CHECK_CTX(c);
  if (replica < 0 || replica >= c->plan.R) return fail(c, HB_EINVAL, "replica out of range");
  select_replica(c, replica);
  return HB_OK;
} HB_CATCH

static int betas_of(hb_ctx* c, const float* T, std::vector<float>& beta) {
  if (!T) return fail(c, HB_EINVAL, "NULL temperature array");
  beta.resize((size_t)c->plan.R);
  for (int32_t r = 0; r < c->plan.R; ++r) {
    const int rc = check_T(c, T[r], &beta[r]);
    if (rc != HB_OK) return rc;
  }
  return HB_OK;
}

int hb_sweep_each(hb_ctx* c, const float* T, int64_t n_sweeps) try {
  HB_CHECK_CTX(c);
  if (n_sweeps < 0) return fail(c, HB_EINVAL, "n_sweeps < 0");
  if (!c->initialised) return fail(c, HB_ESTATE, "spins not initialised");
  std::vector<float> beta;
  int rc = betas_of(c, T, beta);
  if (rc != HB_OK) return rc;
  if (c->plan.R == 1) return hb_sweep(c, T[0], n_sweeps);
  if (n_sweeps == 0) return HB_OK;
  c->cache_valid = c->each_valid = false;
  rc = replica_sweeps(c, beta.data(), n_sweeps, nullptr);
  if (rc == HB_OK) c->each_valid = true;
  return rc;
} HB_CATCH

int hb_measure_each(hb_ctx* c, double* M, double* E) try {
  HB_CHECK_CTX(c);
  if (!M || !E) return fail(c, HB_EINVAL, "NULL output");
  if (!c->initialised) return fail(c, HB_ESTATE, "spins not initialised");
  if (c->plan.R == 1) return hb_measure(c, M, E);
  if (!c->each_valid) {   // no sweep has just produced them: one pass per replica
    const int32_t keep = c->sel;
    for (int32_t r = 0; r < c->plan.R; ++r) {
      select_replica(c, r);
      const int rc = measure_into(c, c->cached_each() + 4 * (size_t)r);
      if (rc != HB_OK) { select_replica(c, keep); return rc; }
    }
    select_replica(c, keep);
    c->each_valid = true;
  }
  std::vector<double> h((size_t)c->plan.R * 4);
  HB_CUDA(c, cudaMemcpyAsync(h.data(), c->cached_each(), h.size() * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
  HB_CUDA(c, cudaStreamSynchronize(c->stream));
  const double inv = 1.0 / (double)c->plan.n;
  for (int32_t r = 0; r < c->plan.R; ++r) {
    M[3 * r] = h[4 * r] * inv; M[3 * r + 1] = h[4 * r + 1] * inv; M[3 * r + 2] = h[4 * r + 2] * inv;
    E[r] = h[4 * r + 3];
  }
  return HB_OK;
} HB_CATCH

int hb_sweep_series_each(hb_ctx* c, const float* T, int64_t n_sweeps, double* M_series, double* E_series) try {
  HB_CHECK_CTX(c);
  if (n_sweeps < 0 || !M_series || !E_series) return fail(c, HB_EINVAL, "bad series arguments");
  if (!c->initialised) return fail(c, HB_ESTATE, "spins not initialised");
  std::vector<float> beta;
  int rc = betas_of(c, T, beta);
  if (rc != HB_OK) return rc;
  if (c->plan.R == 1) return hb_sweep_series(c, T[0], n_sweeps, M_series, E_series);
  if (n_sweeps > 0) c->cache_valid = c->each_valid = false;
  const int32_t R = c->plan.R;
  std::vector<double> h((size_t)R * kSeriesChunk * 4);
  const double inv = 1.0 / (double)c->plan.n;
  for (int64_t s0 = 0; s0 < n_sweeps; s0 += kSeriesChunk) {
    const int64_t m = n_sweeps - s0 < kSeriesChunk ? n_sweeps - s0 : kSeriesChunk;
    rc = replica_sweeps(c, beta.data(), m, c->series());
    if (rc != HB_OK) return rc;
    HB_CUDA(c, cudaMemcpyAsync(h.data(), c->series(), h.size() * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    HB_CUDA(c, cudaStreamSynchronize(c->stream));
    for (int32_t r = 0; r < R; ++r)
      for (int64_t s = 0; s < m; ++s) {
        const double* q = h.data() + ((size_t)r * kSeriesChunk + (size_t)s) * 4;
        double* Mo = M_series + ((size_t)r * (size_t)n_sweeps + (size_t)(s0 + s)) * 3;
        Mo[0] = q[0] * inv; Mo[1] = q[1] * inv; Mo[2] = q[2] * inv;
        E_series[(size_t)r * (size_t)n_sweeps + (size_t)(s0 + s)] = q[3];
      }
  }
  return HB_OK;
} HB_CATCH

// ---- slabs (include/hb.h) -------------------------------------------------------------------
// Local plane z_l holds global plane slab_z0 + z_l - 1 and slab_z0 is even, so the parity of a local plane is the
// opposite of its global one: the sites of GLOBAL colour g are the local colour plane 1 - g.
int hb_slab_pass(hb_ctx* c, float T, int32_t colour) try {
  HB_CHECK_CTX(c);
  if (c->slab_Lz <= 0 && c->plan.part_total <= 0) return fail(c, HB_ESTATE, "not a slab or part context");
  if (colour < 0 || colour >= c->n_colours) return fail(c, HB_EINVAL, "colour: 0 .. colours - 1 (sc: 0 or 1)");
  if (!c->initialised) return fail(c, HB_ESTATE, "spins not initialised");
  float beta;
  int rc = check_T(c, T, &beta);
  if (rc != HB_OK) return rc;
  c->cache_valid = false;
  if (c->plan.part_total > 0) {   // a part of a neighbour table: the own sites of this colour
    rc = one_colour(c, colour, params(c, beta), Diag{nullptr, nullptr});
    if (rc != HB_OK) return rc;
    c->attempts += (uint64_t)(c->colour_begin[colour + 1] - c->colour_begin[colour]);
    return HB_OK;
  }
  if (c->plan.engine == ENGINE_BRAVAIS) {   // colour = basis index, whatever the slab's offset
    rc = one_colour(c, colour, params(c, beta), Diag{nullptr, nullptr});
    if (rc != HB_OK) return rc;
    c->attempts += (uint64_t)c->br.nc - 2ull * (uint64_t)c->br.Lx * c->br.Ly;
    return HB_OK;
  }
  if (c->sc.flag_in) c->sc.stamp = ++c->slab_stamp;   // neighbour flags: this is the slab's pass number `stamp`
  rc = one_colour(c, 1 - colour, params(c, beta), Diag{nullptr, nullptr});
  if (rc != HB_OK) return rc;
  c->attempts += (uint64_t)c->sc.Lx * c->sc.Ly * (uint64_t)(c->sc.Lz - 2) / 2;
  return HB_OK;
} HB_CATCH

int hb_slab_next_sweep(hb_ctx* c) try {
  HB_CHECK_CTX(c);
  if (c->slab_Lz <= 0 && c->plan.part_total <= 0) return fail(c, HB_ESTATE, "not a slab or part context");
  c->sweep += 1;
  return HB_OK;
} HB_CATCH

// ---- parts of a neighbour table: the two halves of the exchange step ---------------------------------------------------------
static int part_move(hb_ctx* c, const int32_t* ids, int64_t count, float* packed, bool gather) {
  HB_CHECK_CTX(c);
  if (c->plan.engine != ENGINE_CSR) return fail(c, HB_ESTATE, "hb_part_gather / hb_part_scatter: neighbour-table contexts (HB_CSR, or per-site anisotropy)");
  if (count < 0 || count > c->plan.n || (count > 0 && (!ids || !packed))) return fail(c, HB_EINVAL, "hb_part_gather / hb_part_scatter: 0 <= count <= n_sites, device arrays");
  if (!c->initialised) return fail(c, HB_ESTATE, "spins not initialised");
  if (count == 0) return HB_OK;
  if (!gather) c->cache_valid = false;
  if (c->plan.ell) {
    if (!c->ell.inv) return fail(c, HB_ESTATE, "hb_part_gather / hb_part_scatter on the ELL engine need a part context (hb_lattice.part_n_total > 0)");
    HB_CUDA(c, launch_part_move_ell(c->stream, c->spins, c->ell.inv, ids, (uint32_t)count, packed, gather));
  } else {
    HB_CUDA(c, launch_part_move_flat(c->stream, c->spins, (uint32_t)c->plan.n, ids, (uint32_t)count, packed, gather));
  }
  c->launches += 1;
  return HB_OK;
}
int hb_part_gather(hb_ctx* c, const int32_t* ids, int64_t count, float* out) try { return part_move(c, ids, count, out, true); } HB_CATCH
int hb_part_scatter(hb_ctx* c, const int32_t* ids, int64_t count, const float* in) try { return part_move(c, ids, count, const_cast<float*>(in), false); } HB_CATCH

int hb_slab_face(hb_ctx* c, int32_t colour, int32_t side, int32_t ghost, size_t offset_floats[3], size_t* count_floats) try {
  HB_CHECK_CTX(c);
  if (c->slab_Lz <= 0) return fail(c, HB_ESTATE, "not a slab context");
  if (colour < 0 || colour >= c->n_colours || ((side | ghost) & ~1)) return fail(c, HB_EINVAL, "colour: 0 .. colours - 1; side, ghost: 0 or 1");
  if (!offset_floats || !count_floats) return fail(c, HB_EINVAL, "NULL output");
  if (c->plan.engine == ENGINE_BRAVAIS) {   // one cell plane of sublattice `colour`: a contiguous run per component
    const size_t plane = (size_t)c->br.Lx * c->br.Ly;
    const int32_t z = side == 0 ? (ghost ? 0 : 1) : (ghost ? c->br.Lz - 1 : c->br.Lz - 2);
    for (int k = 0; k < 3; ++k) offset_floats[k] = (size_t)k * c->br.n + (size_t)colour * c->br.nc + (size_t)z * plane;
    *count_floats = plane;
    return HB_OK;
  }
  const size_t plane = (size_t)c->sc.Ly * c->sc.H;   // sites of one colour in a z-plane: one contiguous run per component
  const int32_t z = side == 0 ? (ghost ? 0 : 1) : (ghost ? c->sc.Lz - 1 : c->sc.Lz - 2);
  for (int k = 0; k < 3; ++k)
    offset_floats[k] = (size_t)k * c->sc.n + (size_t)(1 - colour) * c->sc.half + (size_t)z * plane;
  *count_floats = plane;
  return HB_OK;
} HB_CATCH

int hb_slab_set_peer(hb_ctx* c, int32_t side, void* peer_spins, int32_t peer_Lz) try {
  HB_CHECK_CTX(c);
  if (c->slab_Lz <= 0) return fail(c, HB_ESTATE, "not a slab context");
  if (c->plan.engine != ENGINE_SC) return fail(c, HB_EINVAL, "peer stores exist for simple cubic slabs; bcc / fcc slabs exchange faces (hb_slab_face)");
  if (side != 0 && side != 1) return fail(c, HB_EINVAL, "side: 0 or 1");
  if (peer_spins && (peer_Lz < 2 || (peer_Lz & 1) || (int64_t)c->sc.Lx * c->sc.Ly * ((int64_t)peer_Lz + 2) > 0xFFFFFFFFll))
    return fail(c, HB_EINVAL, "peer_Lz: the neighbour's number of own planes (even, >= 2)");
  const uint32_t plane = (uint32_t)c->sc.Ly * (uint32_t)c->sc.H;   // one colour of one z-plane
  c->sc.peer[side] = static_cast<float*>(peer_spins);
  c->sc.peer_n[side] = peer_spins ? (uint32_t)((int64_t)c->sc.Lx * c->sc.Ly * (peer_Lz + 2)) : 0u;
  c->sc.peer_half[side] = c->sc.peer_n[side] / 2;
  // my low face is the lower neighbour's high ghost plane (its local plane peer_Lz + 1); my high face the upper one's plane 0
  c->sc.peer_zoff[side] = (peer_spins && side == 0) ? (uint32_t)(peer_Lz + 1) * plane : 0u;
  // the neighbour's flag words sit behind its spins: my low side is its upper neighbour (its word 1), my high side its lower (word 0)
  c->sc.flag_out[side] = peer_spins ? reinterpret_cast<uint32_t*>(static_cast<float*>(peer_spins) + 3 * (size_t)c->sc.peer_n[side]) + (side == 0 ? 1 : 0)
                                    : nullptr;
  if (!peer_spins) c->sc.flag_in = nullptr;   // flags need peer stores on both sides
  return HB_OK;
} HB_CATCH

int hb_sweep_count(hb_ctx* c, uint64_t* out) try {
  if (!c || !out) return HB_EINVAL;
  *out = c->sweep;
  return HB_OK;
} HB_CATCH

int hb_set_sweep_count(hb_ctx* c, uint64_t value) try {
  if (!c) return HB_EINVAL;
  c->sweep = value;
  return HB_OK;
} HB_CATCH

int hb_get_colouring(hb_ctx* c, int32_t* colour, int32_t* n_colours) try {
  HB_CHECK_CTX(c);
  if (c->slab_Lz > 0) return fail(c, HB_ESTATE, "slab context: the colour of a site is (x + y + z) mod 2 in global coordinates");
  if (n_colours) *n_colours = c->n_colours;
  if (!colour) return HB_OK;
  if (c->plan.engine == ENGINE_SC) {
    for (int32_t z = 0; z < c->Lz; ++z)
      for (int32_t y = 0; y < c->Ly; ++y)
        for (int32_t x = 0; x < c->Lx; ++x) colour[((int64_t)z * c->Ly + y) * c->Lx + x] = (x + y + z) & 1;
  } else if (c->plan.engine == ENGINE_BRAVAIS) {
    for (int64_t i = 0; i < c->plan.n; ++i) colour[i] = (int32_t)(i / c->br.nc);
  } else {
    std::memcpy(colour, c->colour_host.data(), c->colour_host.size() * sizeof(int32_t));
  }
  return HB_OK;
} HB_CATCH

int hb_counters(hb_ctx* c, uint64_t* kernel_launches, uint64_t* attempts) try {
  if (!c) return HB_EINVAL;
  if (kernel_launches) *kernel_launches = c->launches;
  if (attempts) *attempts = c->attempts;
  return HB_OK;
} HB_CATCH

int hb_sweep_paper_scheme(hb_ctx* c, float T, int64_t n_mcs, int32_t n_per_block) try {
  HB_CHECK_CTX(c);
  if (c->plan.engine != ENGINE_SC || c->slab_Lz > 0 || c->plan.R > 1) return fail(c, HB_EINVAL, "hb_sweep_paper_scheme: a whole simple cubic lattice without replicas");
  if (n_mcs < 0 || n_per_block < 1 || n_per_block > 65536 || c->plan.n % n_per_block) return fail(c, HB_EINVAL, "hb_sweep_paper_scheme: n_mcs >= 0, 1 <= n_per_block <= 65536 dividing the number of sites");
  if (!c->initialised) return fail(c, HB_ESTATE, "spins not initialised");
  float beta;
  const int rc = check_T(c, T, &beta);
  if (rc != HB_OK) return rc;
  if (n_mcs > 0) c->cache_valid = false;
  SweepParams p = params(c, beta);
  for (int64_t s = 0; s < n_mcs; ++s) {
    for (int32_t k = 0; k < n_per_block; ++k) {   // one MCS = N attempts = n_per_block steps of N / n_per_block attempts
      const uint64_t step = c->sweep * 65536ull + (uint64_t)k;
      p.sweep_lo = (uint32_t)step; p.sweep_hi = (uint32_t)(step >> 32);
      HB_CUDA(c, launch_paper_step(c->stream, c->spins, c->sc, p, (uint32_t)n_per_block, c->counters()));
    }
    c->launches += (uint64_t)n_per_block;
    c->sweep += 1;
    c->attempts += (uint64_t)c->plan.n;
    c->stat_attempts += (uint64_t)c->plan.n;
  }
  return HB_OK;
} HB_CATCH

int hb_probe_sc_l2(hb_ctx* c, float T, int64_t n_sweeps, int32_t planes, double* updates_per_second) try {
  HB_CHECK_CTX(c);
  if (!updates_per_second || n_sweeps < 1 || n_sweeps > 100000) return fail(c, HB_EINVAL, "hb_probe_sc_l2: 1 <= n_sweeps <= 100000, non-NULL output");
  if (c->plan.engine != ENGINE_SC || c->slab_Lz > 0 || c->plan.R > 1 || !sc_ws_variant_supported(c->sc, 4) || planes < 2 ||
      (planes & (planes - 1)) || planes > c->sc.Lz)
    return fail(c, HB_EINVAL, "hb_probe_sc_l2: a whole simple cubic lattice with rows of 8..472 sites (Lx % 8 == 0), planes a power of two in [2, Lz]");
  if (!c->initialised) return fail(c, HB_ESTATE, "spins not initialised");
  float beta;
  int rc = check_T(c, T, &beta);
  if (rc != HB_OK) return rc;
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  HB_CUDA(c, cudaEventCreate(&e0));
  if (cudaEventCreate(&e1) != cudaSuccess) { cudaEventDestroy(e0); return fail(c, HB_ECUDA, "cudaEventCreate"); }
  c->cache_valid = c->each_valid = false;
  c->initialised = false;   // the folded addresses leave the lattice in no meaningful state
  SweepParams p = params(c, beta);
  cudaError_t e = cudaSuccess;
  for (int64_t s = -2; s < n_sweeps && e == cudaSuccess; ++s) {   // two untimed sweeps first
    if (s == 0) e = cudaEventRecord(e0, c->stream);
    for (int colour = 0; colour < 2 && e == cudaSuccess; ++colour)
      e = launch_sweep_sc_ws_alias(c->stream, c->spins, c->sc, c->n_sms, c->ws_sched(), p, colour, planes);
    p.sweep_lo += 1;
    c->launches += 2;
  }
  if (e == cudaSuccess) e = cudaEventRecord(e1, c->stream);
  if (e == cudaSuccess) e = cudaEventSynchronize(e1);
  float ms = 0.0f;
  if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  if (e != cudaSuccess) return fail(c, HB_ECUDA, std::string("hb_probe_sc_l2: ") + cudaGetErrorString(e));
  *updates_per_second = (double)c->plan.n * (double)n_sweeps / ((double)ms * 1e-3);
  return HB_OK;
} HB_CATCH

int hb_stats(hb_ctx* c, uint64_t* attempts, uint64_t* accepts) try {
  HB_CHECK_CTX(c);
  if (!attempts || !accepts) return fail(c, HB_EINVAL, "NULL output");
  unsigned long long acc = 0;
  HB_CUDA(c, cudaMemcpyAsync(&acc, c->counters(), sizeof acc, cudaMemcpyDeviceToHost, c->stream));
  HB_CUDA(c, cudaStreamSynchronize(c->stream));
  *attempts = c->stat_attempts;
  *accepts = (uint64_t)acc;
  return HB_OK;
} HB_CATCH

int hb_set_option(hb_ctx* c, const char* name, int64_t value) try {
  HB_CHECK_CTX(c);
  if (!name) return HB_EINVAL;
  const std::string s(name);
  c->g_dirty[0] = c->g_dirty[1] = true;   // the cached graphs were captured with the old settings
  if (s == "graph") {
    if (value < -1 || value > 1) return fail(c, HB_EINVAL, "graph: -1 auto, 0 off, 1 on");
    c->graph_mode = (int)value;
    return HB_OK;
  }
  if (s == "sc_coop") {
    if (value < -1 || value > 2)
      return fail(c, HB_EINVAL, "sc_coop: -1 auto (one block when it fits), 0 off, 1 one block else cooperative grid, 2 cooperative grid");
    c->sc_coop = (int)value;
    return HB_OK;
  }
  if (s == "fused_measure") {
    if (value != 0 && value != 1) return fail(c, HB_EINVAL, "fused_measure: 0 or 1");
    c->fused_measure = value != 0;
    return HB_OK;
  }
  if (s == "pdl") {
    if (value < 0 || value > 2) return fail(c, HB_EINVAL, "pdl: 0 (off), 1 (the next launch comes in as blocks exit), 2 (as soon as every block has started)");
    c->pdl = (int)value;
    c->g_dirty[0] = c->g_dirty[1] = true;   // captured launches carry the attribute
    return HB_OK;
  }
  if (s == "slab_flags") {
    if (value != 0 && value != 1) return fail(c, HB_EINVAL, "slab_flags: 0 or 1");
    if (value == 1 && (c->slab_Lz <= 0 || !c->sc.peer[0] || !c->sc.peer[1] || !sc_ws_supported(c->sc)))
      return fail(c, HB_EINVAL, "slab_flags: a slab context with hb_slab_set_peer on both sides and rows the warp-specialised kernel takes (Lx % 8 == 0, Lx <= 512)");
    c->sc.flag_in = value ? c->slab_flags() : nullptr;
    c->sc.bnd_count = value ? c->slab_bnd_count() : nullptr;
    if (value && c->sc_kernel == 0) c->sc_kernel = 1;   // the flag protocol is part of the warp-specialised kernel
    return HB_OK;
  }
  if (s == "br_kernel" || s == "br_zt") {
    if (c->plan.engine != ENGINE_BRAVAIS) return fail(c, HB_EINVAL, "option valid for bcc / fcc lattices only");
    if (s == "br_kernel") {
      if (value < 0 || value > 2 || (value >= 1 && !bravais_ws_supported(c->br)))
        return fail(c, HB_EINVAL, "br_kernel: 0 (direct), 1 (warp-specialised; needs Lx % 4 == 0 and Lx <= 256), 2 (the same, all colour passes of several sweeps in one launch)");
      c->br_kernel = (int)value;
    } else {
      if (value < 0 || value > c->br.Lz) return fail(c, HB_EINVAL, "br_zt: 1..Lz planes per chunk, 0 = automatic");
      c->br_zt = (int)value;
    }
    clamp_bravais_ws(c);
    return HB_OK;
  }
  if (s == "csr_block") {
    if (value < 32 || value > 256 || value % 32) return fail(c, HB_EINVAL, "csr_block: multiple of 32 in [32,256]");
    c->csr_block = (int)value;
    return HB_OK;
  }
  if (c->plan.engine == ENGINE_CSR) return fail(c, HB_EINVAL, "option not valid for this lattice");
  const bool is_sc = c->plan.engine == ENGINE_SC;
  if (!is_sc && (s == "sc_fused_sweeps" || s == "sc_fused_lag" || s == "sc_ws_ctas")) {   // shared with the bcc / fcc warp-specialised kernel
    if (s == "sc_fused_sweeps") { if (value < 1 || value > 16) return fail(c, HB_EINVAL, "sc_fused_sweeps: 1..16 sweeps per launch"); c->fused_sweeps = (int)value; }
    else if (s == "sc_fused_lag") { if (value < 3 || value > 64) return fail(c, HB_EINVAL, "sc_fused_lag: 3..64 rounds between two colour passes"); c->fused_lag = (int)value; }
    else { if (value < 1 || value > 4096) return fail(c, HB_EINVAL, "sc_ws_ctas: 1..4096"); c->n_sms = (int)value; }
    clamp_bravais_ws(c);
    return HB_OK;
  }
  if (!is_sc && (s == "sc_kernel" || s == "sc_prefetch" || s == "sc_linear" || s == "sc_ws_zt" || s == "sc_ws_variant" || s == "sc_fused_zt"))
    return fail(c, HB_EINVAL, "option valid for the simple cubic lattice only");
  const int32_t rowH = is_sc ? c->sc.H : c->br.Lx, rowLz = is_sc ? c->sc.Lz : c->br.Lz;
  if (s == "sc_kernel") {
    if (value == 2 && 2 * c->fused_sweeps * sc_ws_fused_chunks(c->sc, c->fused_zt) > kWsDoneWords) c->fused_sweeps = 1;
    if (value != 0 && !(value == 1 && sc_ws_supported(c->sc)) &&
        !(value == 2 && sc_ws_fused_supported(c->sc, c->ws_variant) && 2 * c->fused_sweeps * sc_ws_fused_chunks(c->sc, c->fused_zt) <= kWsDoneWords))
      return fail(c, HB_EINVAL, "sc_kernel: 0 (direct), 1 (warp-specialised; needs Lx % 8 == 0 and Lx <= 512) or 2 (the same with all colour "
                                "passes of several sweeps in one launch; whole lattices, sc_ws_variant 2, 4 or 5)");
    if (value == 0 && c->sc.flag_in) return fail(c, HB_EINVAL, "sc_kernel: the neighbour flags of this slab (slab_flags) need the warp-specialised kernel");
    c->sc_kernel = (int)value;
    return HB_OK;
  }
  if (s == "sc_fused_sweeps" || s == "sc_fused_lag" || s == "sc_fused_zt") {
    if (s == "sc_fused_sweeps") { if (value < 1 || value > 16) return fail(c, HB_EINVAL, "sc_fused_sweeps: 1..16 sweeps per launch"); c->fused_sweeps = (int)value; }
    else if (s == "sc_fused_lag") { if (value < 3 || value > 64) return fail(c, HB_EINVAL, "sc_fused_lag: 3..64 rounds between two colour passes"); c->fused_lag = (int)value; }
    else { if (value < 1 || value > c->sc.Lz) return fail(c, HB_EINVAL, "sc_fused_zt: 1..Lz planes per chunk"); c->fused_zt = (int)value; }
    if (2 * c->fused_sweeps * sc_ws_fused_chunks(c->sc, c->fused_zt) > kWsDoneWords) {
      c->fused_sweeps = 1; c->fused_zt = 8;
      return fail(c, HB_EINVAL, "sc_fused_*: passes x chunks exceeds the progress words of the workspace");
    }
    return HB_OK;
  }
  if (s == "sc_ws_zt") {
    if (value < 0 || value > c->sc.Lz) return fail(c, HB_EINVAL, "sc_ws_zt: 1..Lz, or 0 = balanced over the persistent CTAs");
    c->ws_zt = (int)value;
    return HB_OK;
  }
  if (s == "sc_ws_variant") {
    if (!sc_ws_variant_supported(c->sc, (int)value))
      return fail(c, HB_EINVAL, "sc_ws_variant: 0 (4-row tiles, 2 CTAs per SM), 1 (8-row tiles, 1 CTA per SM), 2 (4-row tiles, 3 CTAs per SM), "
                                "3 (16-row tiles, 1 CTA per SM; rows of up to 248 floats), 4 (7-row tiles, 2 CTAs per SM; rows of up to 236 floats), "
                                "5 (8-row tiles at a 512-byte pitch, 3 CTAs per SM; rows of up to 128 floats)");
    c->ws_variant = (int)value;
    if (c->sc_kernel == 2 && !sc_ws_fused_supported(c->sc, c->ws_variant)) c->sc_kernel = 1;
    return HB_OK;
  }
  if (s == "sc_ws_ctas") {
    if (value < 1 || value > 4096) return fail(c, HB_EINVAL, "sc_ws_ctas: 1..4096");
    c->n_sms = (int)value;
    return HB_OK;
  }
  ScTile t = c->tile;
  if (s == "sc_v") {
    if (!(value == 1 || value == 2 || value == 4) || rowH % value)
      return fail(c, HB_EINVAL, "sc_v: 1, 2 or 4 dividing the row length (Lx/2 for sc, Lx for bcc/fcc)");
    t.V = (int)value;
    if (t.JX > rowH / t.V) t.JX = rowH / t.V;
  } else if (s == "sc_jx") t.JX = (int)value;
  else if (s == "sc_ty") t.TY = (int)value;
  else if (s == "sc_zt") t.ZT = (int)value;
  else if (s == "sc_prefetch") { if (value < 0 || value > 3) return fail(c, HB_EINVAL, "sc_prefetch: 0..3"); t.PF = (int)value; }
  else if (s == "sc_linear") {
    if (value != 0 && (value < 32 || value > 256 || value % 32)) return fail(c, HB_EINVAL, "sc_linear: 0 or a multiple of 32 up to 256");
    t.LIN = (int)value;
  }
  else return fail(c, HB_EINVAL, "unknown option");
  const int64_t max_threads = (is_sc && t.V == 4) ? 1024 : 256;   // the big-block variants exist for sc, V = 4
  if (t.JX < 1 || t.TY < 1 || t.ZT < 1 || (int64_t)t.JX * t.TY > max_threads || t.ZT > rowLz)
    return fail(c, HB_EINVAL, "sc tile: JX, TY, ZT >= 1, JX*TY <= 256 (1024 for sc with V = 4), ZT <= Lz");
  c->tile = t;
  return HB_OK;
} HB_CATCH

int hb_get_option(hb_ctx* c, const char* name, int64_t* value) try {
  if (!c || !name || !value) return HB_EINVAL;
  const std::string s(name);
  if (s == "csr_block") *value = c->csr_block;
  else if (s == "pdl") *value = c->pdl;
  else if (s == "fused_measure") *value = c->fused_measure ? 1 : 0;
  else if (s == "sc_coop") *value = c->sc_coop;
  else if (s == "graph") *value = c->graph_mode;
  else if (s == "graph_active") *value = graph_wanted(c) ? 1 : 0;
  else if (s == "coop_active") *value = coop_mode(c) != 0 ? 1 : 0;
  else if (s == "sc_v") *value = c->tile.V;
  else if (s == "sc_jx") *value = c->tile.JX;
  else if (s == "sc_ty") *value = c->tile.TY;
  else if (s == "sc_zt") *value = c->tile.ZT;
  else if (s == "sc_prefetch") *value = c->tile.PF;
  else if (s == "sc_linear") *value = c->tile.LIN;
  else if (s == "engine") *value = c->plan.engine;
  else if (s == "ell") *value = c->plan.ell ? 1 : 0;
  else if (s == "sc_kernel") *value = c->sc_kernel;
  else if (s == "sc_ws_zt") *value = c->ws_zt;
  else if (s == "sc_ws_ctas") *value = c->n_sms;
  else if (s == "sc_ws_variant") *value = c->ws_variant;
  else if (s == "sc_fused_sweeps") *value = c->fused_sweeps;
  else if (s == "sc_fused_lag") *value = c->fused_lag;
  else if (s == "sc_fused_zt") *value = c->fused_zt;
  else if (s == "slab_flags") *value = c->sc.flag_in ? 1 : 0;
  else if (s == "br_kernel") *value = c->br_kernel;
  else if (s == "br_zt") *value = c->br_zt;
  else return HB_EINVAL;
  return HB_OK;
} HB_CATCH

int hb_lattice_fcc_sphere(int32_t R, float K_core, const float e_core[3], float K_surf, int32_t colouring,
                          hb_lattice* out, int32_t** xyz_out) try {
  if (!out || !e_core || R < 0 || R > 200 || (colouring != 0 && colouring != 1)) return HB_EINVAL;
  HostCsr g;
  std::vector<int32_t> xyz;
  build_fcc_sphere_csr(R, g, xyz);
  if (colouring == 0) {
    greedy_first_fit(g);
  } else {
    for (int64_t i = 0; i < g.n; ++i) g.colour[i] = (xyz[3 * i] & 1) * 2 + (xyz[3 * i + 1] & 1);
    g.n_colours = 4;
    if (g.n == 1) g.n_colours = 1;
  }
  std::memset(out, 0, sizeof *out);
  const size_t n = (size_t)g.n, nnz = g.col.size();
  int64_t* rp = static_cast<int64_t*>(std::malloc((n + 1) * sizeof(int64_t)));
  int32_t* ci = static_cast<int32_t*>(std::malloc((nnz ? nnz : 1) * sizeof(int32_t)));
  int32_t* cc = static_cast<int32_t*>(std::malloc(n * sizeof(int32_t)));
  float* Ks = static_cast<float*>(std::malloc(n * sizeof(float)));
  float* es = static_cast<float*>(std::malloc(3 * n * sizeof(float)));
  int32_t* xo = xyz_out ? static_cast<int32_t*>(std::malloc(3 * n * sizeof(int32_t))) : nullptr;
  if (!rp || !ci || !cc || !Ks || !es || (xyz_out && !xo)) {
    std::free(rp); std::free(ci); std::free(cc); std::free(Ks); std::free(es); std::free(xo);
    return HB_ENOMEM;
  }
  std::memcpy(rp, g.row_ptr.data(), (n + 1) * sizeof(int64_t));
  if (nnz) std::memcpy(ci, g.col.data(), nnz * sizeof(int32_t));
  std::memcpy(cc, g.colour.data(), n * sizeof(int32_t));
  for (size_t i = 0; i < n; ++i) {
    const bool core = (rp[i + 1] - rp[i]) == 12;
    if (core) {
      Ks[i] = K_core; es[3 * i] = e_core[0]; es[3 * i + 1] = e_core[1]; es[3 * i + 2] = e_core[2];
    } else {
      const double X = xyz[3 * i], Y = xyz[3 * i + 1], Z = xyz[3 * i + 2];
      const double rr = std::sqrt(X * X + Y * Y + Z * Z);
      Ks[i] = K_surf;
      es[3 * i] = rr > 0 ? (float)(X / rr) : 0.0f;
      es[3 * i + 1] = rr > 0 ? (float)(Y / rr) : 0.0f;
      es[3 * i + 2] = rr > 0 ? (float)(Z / rr) : 1.0f;
    }
  }
  if (xo) { std::memcpy(xo, xyz.data(), 3 * n * sizeof(int32_t)); *xyz_out = xo; }
  out->kind = HB_CSR; out->n_sites = g.n; out->row_ptr = rp; out->col_idx = ci;
  out->n_colours = g.n_colours; out->colour = cc; out->K_site = Ks; out->e_site = es;
  return HB_OK;
} HB_CATCH

int hb_lattice_free(hb_lattice* lat) try {
  if (!lat) return HB_OK;
  std::free(const_cast<int64_t*>(lat->row_ptr));
  std::free(const_cast<int32_t*>(lat->col_idx));
  std::free(const_cast<int32_t*>(lat->colour));
  std::free(const_cast<float*>(lat->K_site));
  std::free(const_cast<float*>(lat->e_site));
  std::memset(lat, 0, sizeof *lat);
  return HB_OK;
} HB_CATCH

const char* hb_strerror(int status) {
  switch (status) {
    case HB_OK: return "ok";
    case HB_EINVAL: return "invalid argument";
    case HB_ENOMEM: return "out of memory or buffer too small";
    case HB_ECUDA: return "CUDA error";
    case HB_ESTATE: return "call out of order";
    default: return "unknown status";
  }
}

const char* hb_error_detail(hb_ctx* c) { return c ? c->detail.c_str() : ""; }

}  // extern "C"
