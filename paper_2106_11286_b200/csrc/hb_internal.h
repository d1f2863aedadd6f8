// hb_internal.h -- host-side declarations shared by hb_api.cpp, hb_lattice.cpp and hb_kernels.cu.
#pragma once
#include <cstddef>
#include <cstdint>
#include <string>
#include <vector>

#include <cuda_runtime.h>

namespace hb {

// parameters of one colour pass (passed by value to the kernels)
struct SweepParams {
  float J, K, ex, ey, ez, beta;
  uint32_t seed_lo, seed_hi, sweep_lo, sweep_hi;
  // Replayed launches (CUDA graph) cannot carry the sweep counter in their parameters: with
  // sweep_dev != nullptr the counter is *sweep_dev + sweep_lo (sweep_lo = index of the sweep inside the graph)
  const unsigned long long* sweep_dev;
  // launch the colour kernel with programmatic stream serialisation: its blocks may become resident
  // while the previous kernel of the stream drains; every colour kernel waits (griddepcontrol.wait, in resolve_sweep)
  // for that kernel to complete before it touches memory
  int32_t pdl;
};

// kern<<<grid, block, smem, st>>>(args...), with the programmatic-serialisation attribute when pdl is set
template <class... KArgs, class... Args>
inline cudaError_t launch_colour_kernel(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, bool pdl,
                                        Args&&... args) {
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr; cfg.numAttrs = pdl ? 1 : 0;
  return cudaLaunchKernelEx(&cfg, kern, KArgs(args)...);
}

// simple cubic, colour-split storage
struct ScLayout {
  int32_t Lx, Ly, Lz;
  int32_t H;        // Lx/2: sites of one colour per x-row
  uint32_t half;    // N/2: sites per colour
  uint32_t n;       // N
  // slab of a larger lattice (include/hb.h, hb_lattice.slab_Lz): planes 0 and Lz-1 are ghost planes, the Philox site id
  // of local site s is s + site_base (mod 2^32); both 0 for a whole lattice
  uint32_t site_base;
  int32_t ghost;
  // slab with peer stores (hb_slab_set_peer): a thread that stores an updated spin of its first / last own plane also
  // stores it into the ghost plane of the z-neighbour's spins buffer (peer memory over NVLink, or the same device):
  // peer[side] = that buffer (x component), peer_n / peer_half its component and colour strides, peer_zoff the offset
  // of its ghost plane; side 0 = my low face -> the lower neighbour's high ghost plane, 1 = the other way
  float* peer[2];
  uint32_t peer_n[2], peer_half[2], peer_zoff[2];
  // Neighbour flags instead of a barrier between two colour passes (hb_set_option "slab_flags", warp-specialised kernel, peer
  // stores on both sides).  Pass number `stamp` (1, 2, ...) of a slab takes its two boundary chunks
  // first; a boundary tile waits until the neighbour on that side has finished ITS boundary chunk of pass stamp - 1
  // (flag_in[side] >= stamp - 1: the ghost plane it reads is complete, and the neighbour no longer reads the ghost plane
  // this pass stores into); the warp that finishes the last tile of a boundary chunk writes `stamp` into the neighbour's
  // flag (flag_out[side], peer memory, release at system scope).  flag_in: two words behind this slab's spins;
  // bnd_count: two words of its workspace; nullptr = off.
  uint32_t* flag_in;
  uint32_t* flag_out[2];
  uint32_t* bnd_count;
  uint32_t stamp;
};

// launch shape of the sc kernels: a block is JX x TY threads, each thread owns V
// consecutive same-colour sites of one x-row and marches ZT planes in z
struct ScTile {
  int32_t V, JX, TY, ZT;
  int32_t PF;   // software prefetch of the next z-plane: 0 none, 1 L2, 2 L1, 3 touch
  int32_t LIN;  // 0: JX x TY tile; > 0: threads per block of the linear (y, j) mapping (full warps); < 0: one block, (z, y, j)
};

// periodic Bravais lattice with a basis (bcc: 2 sublattices, fcc: 4), canonical storage:
// sublattice b is an Lx x Ly x Lz array at offset b*nc of each component plane
enum { BR_BCC = 1, BR_FCC = 2 };   // values of hb_kind
struct BrLayout {
  int32_t kind;
  int32_t Lx, Ly, Lz;
  uint32_t nc;      // cells = sites per sublattice
  uint32_t n;       // N
  // slab of a larger lattice along z (include/hb.h, hb_lattice.slab_Lz): cell planes 0 and Lz-1 of every sublattice are
  // ghost planes (staged as neighbours, not updated, not measured); the Philox id of local cell q of sublattice b is
  // b * nc_id + q + cell_base (mod 2^32) with nc_id the cells of the WHOLE lattice.  ghost = 0: nc_id = nc, cell_base = 0.
  int32_t ghost;
  uint32_t nc_id, cell_base;
};

// CSR tables on the device
struct CsrDev {
  uint32_t n;
  uint32_t n_own;           // sites that are attempted and measured: n, or the own sites of a part (the rest are ghosts)
  uint32_t site_base;       // Philox counter word of local site i is i + site_base (a part of a larger table; else 0)
  const int32_t* row_ptr;   // n+1
  const int32_t* col;       // nnz
  const int32_t* list;      // sites sorted by (colour, id)
  const float* K_site;      // n or nullptr
  const float* e_site;      // 3n or nullptr
};

// Neighbour table in colour-major ELL form.  Spins are AoS float4 (x, y, z, 0) in INTERNAL order m
// (sorted by colour, then canonical id); colour c owns m in [begin_c, begin_c + n_c).  Entry k of the
// t-th site of colour c sits at ell[maxdeg*begin_c + k*n_c + t] (consecutive threads read consecutive
// words), holds the internal index of the k-th neighbour in the caller's order, or -1 past the degree.
struct EllDev {
  uint32_t n, maxdeg;
  const int32_t* ell;
  const int32_t* perm;          // internal index -> canonical id (+ site_base: the Philox counter word)
  uint32_t site_base;           // a part of a larger table: global id of local site 0; else 0
  const int32_t* inv;           // canonical id -> internal index (parts only: hb_part_gather / scatter), or nullptr
  const uint32_t* colour_begin; // n_colours + 1 entries (device copy, for the measurement pass)
  int32_t n_colours;
  const float* K;               // per-site anisotropy in internal order, SoA; or nullptr
  const float* ex; const float* ey; const float* ez;
};

// diagnostics of one sweep
struct Diag {
  uint8_t* accept;                  // n bytes (canonical id) or nullptr
  unsigned long long* n_accept;     // or nullptr
};

// measurement fused into a colour pass (sc, two colours): block partials of (sum S, energy terms)
struct Meas {
  double* partials;   // 4 doubles per block of the launch, or nullptr
  int mode;           // 0 off, 1 own spins + anisotropy energy, 2 also the exchange energy (last colour)
  unsigned long long* n_accept = nullptr;   // accepted moves of the pass are added here (hb_stats), one atomic per warp; or nullptr
};

constexpr int kFusedBlocksMax = 16384;   // per colour: larger grids use the separate measurement pass

// ---- kernels (hb_kernels.cu); every launcher returns the launch status -----------------
cudaError_t launch_init_random_sc(cudaStream_t st, float* spins, ScLayout L, uint32_t seed_lo, uint32_t seed_hi);
cudaError_t launch_init_random_flat(cudaStream_t st, float* spins, uint32_t n, uint32_t seed_lo, uint32_t seed_hi, uint32_t site_base = 0);
cudaError_t launch_init_random_bravais(cudaStream_t st, float* spins, BrLayout L, uint32_t seed_lo, uint32_t seed_hi);
cudaError_t launch_fill(cudaStream_t st, float* spins, uint32_t n, float x, float y, float z);
cudaError_t launch_sc_permute(cudaStream_t st, float* dst, const float* src, ScLayout L, bool to_internal);
// one step of the paper's own scheme, emulated (hb_sweep_paper_scheme): p.sweep_lo/hi = the step number
cudaError_t launch_paper_step(cudaStream_t st, float* spins, ScLayout L, SweepParams p, uint32_t n_per_block, unsigned long long* n_accept);
cudaError_t launch_sweep_sc(cudaStream_t st, float* spins, ScLayout L, ScTile t, SweepParams p, int colour, Diag d, Meas m);
// blocks one launch_sweep_sc launch uses with this tile if it can carry the fused measurement, else 0
int sc_fused_blocks(const ScLayout& L, const ScTile& t);
// persistent multi-sweep paths of the sc engine: ONE block when a colour pass fits 1024 threads (N <= 8192), or a
// cooperative grid with a grid-wide barrier per colour.  sc_coop_blocks: virtual blocks of a pass, 0 = unavailable.
// partials must hold 2 x 2 x blocks x 4 doubles; series (4 doubles per sweep) or final_out (4 doubles) may be null
int sc_one_block_threads(const ScLayout& L);
int sc_coop_blocks(const ScLayout& L, const ScTile& t);
// one_block with n_replicas > 1: block r runs replica r (state at spins + 3 N r, key seed + r, beta betas[r] if betas,
// partials + 16 r, series + series_stride r, final_out + 4 r)
cudaError_t launch_sweeps_sc_coop(cudaStream_t st, float* spins, ScLayout L, ScTile t, SweepParams p, uint64_t sweep0, int n_sweeps,
                                  bool one_block, double* partials, double* series, double* final_out,
                                  int n_replicas, const float* betas, uint64_t series_stride, unsigned long long* n_accept);
// warp-specialised persistent sc kernel (hb_sc_ws.cu): grid_cap = CTAs to launch at most (one per SM)
bool sc_ws_supported(const ScLayout& L);
bool sc_ws_variant_supported(const ScLayout& L, int variant);
int sc_ws_blocks(const ScLayout& L, int ZT, int grid_cap, int variant);
cudaError_t launch_sweep_sc_ws(cudaStream_t st, float* spins, ScLayout L, int ZT, int grid_cap, int variant, uint32_t* sched /* 2 device words, zero */,
                               SweepParams p, int colour, Meas m);
// diagnostic (hb_probe_sc_l2): one colour pass of the 7-row variant with the address of plane z folded onto plane z mod planes
cudaError_t launch_sweep_sc_ws_alias(cudaStream_t st, float* spins, ScLayout L, int grid_cap, uint32_t* sched, SweepParams p, int colour, int planes);
// fused launches of the same kernel: n_sweeps whole sweeps = 2 n_sweeps colour passes in ONE launch, tiles
// ordered in rounds with `lag` (>= 3) rounds between two passes; done = kWsDoneWords device words, zero between launches;
// m.mode != 0: the LAST sweep of the launch carries the fused measurement (block partials: one per CTA)
constexpr int kWsDoneWords = 16384;
bool sc_ws_fused_supported(const ScLayout& L, int variant);
int sc_ws_fused_chunks(const ScLayout& L, int ZT);
int sc_ws_fused_blocks(const ScLayout& L, int ZT, int grid_cap, int variant, int n_sweeps);
cudaError_t launch_sweep_sc_ws_fused(cudaStream_t st, float* spins, ScLayout L, int ZT, int lag, int grid_cap, int variant, uint32_t* sched,
                                     uint32_t* done, SweepParams p, int n_sweeps, Meas m);
cudaError_t launch_sweep_csr(cudaStream_t st, float* spins, CsrDev g, uint32_t list_begin, uint32_t list_count,
                             SweepParams p, int block, Diag d);
cudaError_t launch_sweep_ell(cudaStream_t st, float* spins, EllDev g, uint32_t begin, uint32_t count, SweepParams p,
                             int block, Diag d);
cudaError_t launch_measure_ell(cudaStream_t st, const float* spins, EllDev g, SweepParams p, double* partials, double* out);
cudaError_t launch_init_random_perm(cudaStream_t st, float* spins, const int32_t* perm, uint32_t n, uint32_t seed_lo, uint32_t seed_hi, uint32_t site_base = 0);
// exchange step of table parts (hb_part_gather / hb_part_scatter): spins of the listed local sites <-> packed (x, y, z, 0) records.
// ELL engine: AoS state, ids translated through inv; CSR engine: three planes of n floats
cudaError_t launch_part_move_ell(cudaStream_t st, float* spins, const int32_t* inv, const int32_t* ids, uint32_t count, float* packed, bool gather);
cudaError_t launch_part_move_flat(cudaStream_t st, float* spins, uint32_t n, const int32_t* ids, uint32_t count, float* packed, bool gather);
cudaError_t launch_fill_ell(cudaStream_t st, float* spins, uint32_t n, float x, float y, float z);
// component comp of the internal float4 state <- plane[perm[m]] (to_internal) or plane[perm[m]] <- component
cudaError_t launch_permute_ell(cudaStream_t st, float* spins, float* plane, const int32_t* perm, uint32_t n, int comp, bool to_internal);
// warp-specialised persistent bcc / fcc kernel (hb_bravais_ws.cu): `passes` colour passes in one launch, starting with colour
// `first` of the sweep in p (one pass = a plain colour launch); rows of up to 256 cells, Lx a multiple of 4
bool bravais_ws_supported(const BrLayout& L);
int bravais_ws_chunks(const BrLayout& L, int ZT, int grid_cap);
int bravais_ws_blocks(const BrLayout& L, int ZT, int grid_cap, int passes);
cudaError_t launch_sweep_bravais_ws(cudaStream_t st, float* spins, BrLayout L, int ZT, int lag, int grid_cap, uint32_t* sched, uint32_t* done,
                                    SweepParams p, int first, int passes, Meas m);
int bravais_fused_blocks(const BrLayout& L, const ScTile& t);
cudaError_t launch_sweep_bravais(cudaStream_t st, float* spins, BrLayout L, ScTile t, SweepParams p, int colour, Diag d, Meas m);
// measurement: partials must hold kMeasureBlocks*4 doubles; out receives (Mx*N, My*N, Mz*N, E)
constexpr int kMeasureBlocks = 1184;
cudaError_t launch_measure_sc(cudaStream_t st, const float* spins, ScLayout L, int V, SweepParams p, double* partials, double* out);
cudaError_t launch_measure_csr(cudaStream_t st, const float* spins, CsrDev g, SweepParams p, double* partials, double* out);
cudaError_t launch_measure_bravais(cudaStream_t st, const float* spins, BrLayout L, int V, SweepParams p, double* partials, double* out);
cudaError_t launch_reduce_final(cudaStream_t st, const double* partials, int n_blocks, double* out);
// replayed launches: (sum S, E) goes to entry *idx of series, then *idx advances by one
cudaError_t launch_reduce_final_series(cudaStream_t st, const double* partials, int n_blocks, double* series,
                                       unsigned long long* idx);
// *counter = value (add == false) or *counter += value: the device-side sweep counter of replayed launches
cudaError_t launch_set_counter(cudaStream_t st, unsigned long long* counter, unsigned long long value, bool add);

// ---- host lattice tables (hb_lattice.cpp) -------------------------------------------------
struct HostCsr {
  int64_t n = 0;
  std::vector<int64_t> row_ptr;
  std::vector<int32_t> col;
  std::vector<int32_t> colour;
  int32_t n_colours = 0;
};
void build_bcc_csr(int32_t Lx, int32_t Ly, int32_t Lz, HostCsr& out);
void build_fcc_csr(int32_t Lx, int32_t Ly, int32_t Lz, HostCsr& out);
void build_fcc_sphere_csr(int32_t R, HostCsr& out, std::vector<int32_t>& xyz);
void greedy_first_fit(HostCsr& g);
// empty string = valid; otherwise what is wrong
// n_own < n: a part of a larger table: sites n_own .. n-1 are ghosts (empty rows); symmetry is checked among the own sites
std::string validate_csr(int64_t n, const int64_t* row_ptr, const int32_t* col, int64_t n_own = -1);
std::string validate_colouring(int64_t n, const int64_t* row_ptr, const int32_t* col, const int32_t* colour,
                               int32_t n_colours, int64_t n_own = -1);

}  // namespace hb
