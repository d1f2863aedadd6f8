/* hb.h -- C ABI of the B200 Metropolis colour-sweep library (libhb.so).
 *
 * What it computes: the single-spin-update Metropolis sweep of the classical
 * anisotropic Heisenberg model of arXiv 2106.11286,
 *     H = -J sum_<ij> S_i.S_j - sum_i K_i (S_i.e_i)^2          (eq. 1)
 * with |S_i| = 1 (line 40), update rule (i)-(iii) of line 20 (propose a uniformly
 * random orientation, accept if dH <= 0 or P <= exp(-dH/T)), and the
 * magnetisation M = (1/N) sum_i S_i of eq. 2 (line 22) plus the total energy,
 * both reduced on the device.  The random site choice of step (i) is replaced
 * by conflict-free colour-ordered sweeps (reading A3): every site
 * attempts exactly once per sweep, colour by colour, one CUDA kernel per colour.
 *
 * Conventions
 *  - every function returns HB_OK (0) or a negative hb_status; nothing throws,
 *    aborts or prints (a failed host allocation inside the library comes back as
 *    HB_ENOMEM: every entry point catches at the boundary).  hb_strerror() names a status, hb_error_detail() gives
 *    the last message (CUDA error string included) of a context.
 *  - "host" pointers are ordinary CPU memory, "device" pointers are CUDA device
 *    memory of the current device.  The library never frees caller memory.
 *  - spins are three fp32 planes (x, y, z), as in the paper (line 30: "three
 *    one-dimensional arrays").  Host-side spin arrays use the CANONICAL site
 *    order: sc id = (z*Ly + y)*Lx + x; bcc/fcc id = b*Ncell + (z*Ly + y)*Lx + x
 *    with b the basis index; CSR id = the caller's row index.  The device
 *    layout is private to the library.
 *  - a context is not thread-safe; distinct contexts are independent.
 *  - all work is enqueued on the context's CUDA stream; hb_sweep is
 *    asynchronous, every call that returns data to the host synchronises.
 */
#ifndef HB_H_
#define HB_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct hb_ctx hb_ctx;

typedef enum {
  HB_OK = 0,
  HB_EINVAL = -1,  /* bad argument: odd L for sc, T <= 0 or NaN, non-unit axis, asymmetric CSR, improper colouring ... */
  HB_ENOMEM = -2,  /* host or device allocation failed, or a caller buffer is too small */
  HB_ECUDA = -3,   /* a CUDA call failed; sticky for the context */
  HB_ESTATE = -4   /* call order: sweep or measure before the spins were initialised */
} hb_status;

typedef enum {
  HB_SC = 0,   /* simple cubic, periodic, z = 6, 2 colours (x+y+z) mod 2; Lx, Ly, Lz even            */
  HB_BCC = 1,  /* bcc, periodic, 2 sites per conventional cell, z = 8, colour = basis index          */
  HB_FCC = 2,  /* fcc, periodic, 4 sites per conventional cell, z = 12, colour = basis index         */
  HB_CSR = 3   /* arbitrary neighbour table (free-boundary nanostructures), any proper colouring     */
} hb_kind;

/* Lattice description (host memory, read during hb_create only; the caller keeps ownership).
 * Neighbour summation order is part of the arithmetic (fp32 adds do not commute bitwise):
 *   sc : -x,+x,-y,+y,-z,+z
 *   bcc: corner (b=0) of cell (x,y,z): centres of cells (x-1|x, y-1|y, z-1|z), x fastest;
 *        centre (b=1): corners of cells (x|x+1, y|y+1, z|z+1), x fastest
 *   fcc: basis b0 (0,0,0), b1 (0,1/2,1/2), b2 (1/2,0,1/2), b3 (1/2,1/2,0); offsets in doubled
 *        coordinates (+1,+1,0),(+1,-1,0),(-1,+1,0),(-1,-1,0),(+1,0,+1),(+1,0,-1),(-1,0,+1),
 *        (-1,0,-1),(0,+1,+1),(0,+1,-1),(0,-1,+1),(0,-1,-1)
 *   CSR: the order of col_idx within the row.                                                   */
typedef struct {
  int32_t kind;            /* hb_kind */
  int32_t Lx, Ly, Lz;      /* conventional cells per direction (Bravais kinds) */
  /* HB_CSR only: */
  int64_t n_sites;
  const int64_t* row_ptr;  /* n_sites + 1 entries, row_ptr[0] = 0 */
  const int32_t* col_idx;  /* row_ptr[n_sites] entries; symmetric (with multiplicity), no self loops */
  int32_t n_colours;       /* with colour != NULL: number of colours, values 0..n_colours-1 */
  const int32_t* colour;   /* NULL => the library runs greedy first-fit in site order */
  /* any kind, optional per-site anisotropy (canonical order); NULL => the uniform (K, e) of hb_create */
  const float* K_site;     /* n entries */
  const float* e_site;     /* 3n entries, (ex,ey,ez) per site, unit vectors */
  /* independent replicas of the lattice in one context (0 or 1: a single system).  Replica r is the system
   * with Philox key seed + r; more than one needs a simple cubic lattice of at most 8192 sites with Lx a
   * multiple of 8 and uniform anisotropy (each replica runs in one thread block, hb_sweep_each below). */
  int32_t n_replicas;
  /* Slab of a larger periodic sc, bcc or fcc lattice (multi-GPU decomposition along z).
   * slab_Lz = 0: none.  slab_Lz > 0: the context holds planes (of conventional cells) z = slab_z0 .. slab_z0 + Lz - 1 of a
   * lattice of Lx x Ly x slab_Lz cells (sc: Lz, slab_z0, slab_Lz even), plus, for every sublattice, one ghost plane on each
   * side that the caller keeps current (hb_slab_face).  Philox is keyed by the GLOBAL site id, so the slabs together walk the trajectory of the
   * whole lattice bit for bit.  Such a context is driven with hb_slab_pass / hb_slab_next_sweep instead of hb_sweep. */
  int32_t slab_Lz, slab_z0;
  /* Part of a larger neighbour table (HB_CSR; multi-GPU decomposition by ranges of the canonical order).
   * part_n_total = 0: none.  part_n_total > 0: the context holds sites part_first .. part_first + part_n_own - 1 of a table of
   * part_n_total sites as its local sites 0 .. part_n_own - 1, followed by n_sites - part_n_own GHOST sites: copies of
   * other parts' sites that the local rows point to.  Ghost rows are empty; ghosts are never attempted or measured, the caller
   * keeps them current (hb_part_gather on the owner, hb_part_scatter here, after every colour pass).  `colour` is required:
   * the colouring of the WHOLE table restricted to the local sites, ghosts included (checked on the own rows).  Philox is
   * keyed by the global id part_first + local id, so the parts together walk the trajectory of the whole table bit for bit.
   * Such a context is driven with hb_slab_pass / hb_slab_next_sweep like a slab; hb_measure returns its share (M normalised
   * by part_n_total, every bond half at each end); hb_get_spins / hb_set_spins move all n_sites local sites, ghosts included. */
  int64_t part_n_total, part_first, part_n_own;
} hb_lattice;

/* Caller-owned device memory (e.g. torch tensors).  Sizes from hb_sizes().  Both
 * pointers must be 256-byte aligned.  NULL hb_buffers* in hb_create => the library
 * allocates with cudaMalloc and frees in hb_destroy. */
typedef struct {
  void* spins;            /* device, spins_bytes */
  size_t spins_bytes;
  void* workspace;        /* device, workspace_bytes (lattice tables, staging, reduction scratch) */
  size_t workspace_bytes;
  void* cuda_stream;      /* cudaStream_t; NULL => the legacy default stream */
} hb_buffers;

/* Number of sites and the device bytes a context for this lattice needs. */
int hb_sizes(const hb_lattice* lat, int64_t* n_sites, size_t* spins_bytes, size_t* workspace_bytes);

/* Build a context: validates the lattice, colours it, uploads its tables.
 * J: exchange; (K, e): uniform uniaxial anisotropy, e a unit vector (|e|^2 within 1e-5 of 1);
 * seed: key of the counter-based Philox4x32-10 stream.  The random numbers of the attempt
 * at site i in sweep s are Philox(counter = (i, 0, s_lo, s_hi), key = (seed_lo, seed_hi)),
 * identical on any device and in the CPU oracle. */
int hb_create(hb_ctx** out, const hb_lattice* lat, float J, float K, const float e[3], uint64_t seed,
              const hb_buffers* bufs);
int hb_destroy(hb_ctx* ctx);

/* Initial state.  random: S_i = sphere(Philox(counter = (i, 1, 0, 0))): uniform unit vectors.
 * aligned: S_i = dir (a unit vector).  set/get: host arrays of n floats each, canonical order. */
int hb_init_random(hb_ctx* ctx);
int hb_init_aligned(hb_ctx* ctx, const float dir[3]);
int hb_set_spins(hb_ctx* ctx, const float* sx, const float* sy, const float* sz);
int hb_get_spins(hb_ctx* ctx, float* sx, float* sy, float* sz);
/* The same upload in two halves, so that the copy of the NEXT state overlaps the sweeps of the current one (a run that
 * feeds a fresh state every step): hb_stage_spins starts the host->device copy of three canonical arrays (pinned host
 * memory, or the copy is not asynchronous) into a library-owned upload area of 3 n floats on a stream of its own and returns
 * at once; hb_commit_spins waits for that copy, then makes the staged state the context's state, in stream order with the
 * sweeps before and after it.  The host arrays must stay untouched until hb_commit_spins has returned.  One staged state
 * at a time: a second hb_stage_spins before the commit returns HB_ESTATE.  Whole lattices without replicas. */
int hb_stage_spins(hb_ctx* ctx, const float* sx, const float* sy, const float* sz);
int hb_commit_spins(hb_ctx* ctx);

/* n_sweeps Metropolis sweeps at temperature T (units of J/k_B, T > 0, +inf allowed).
 * One sweep = one attempt at every site, colours in ascending order.  Asynchronous.
 * The sweep counter (the Philox counter words 2,3) advances by n_sweeps and is never reset.
 * How the launches are issued (one kernel per colour, a replayed CUDA graph of 8 sweeps on small
 * lattices, one persistent block on tiny ones) does not change a bit of the result. */
int hb_sweep(hb_ctx* ctx, float T, int64_t n_sweeps);

/* M[3] = (1/N) sum_i S_i (eq. 2) and E = total energy of eq. 1 (each bond once), accumulated
 * in fp64 from fp32 per-site terms -0.5 J (S_i.h_i) - K_i (S_i.e_i)^2.  Synchronises.
 * On the sc, bcc and fcc engines the last sweep of hb_sweep has already reduced both (each bond
 * charged once, at its higher-colour end; same tolerances), so this call only copies 32 bytes;
 * after hb_set_spins / hb_init_* / hb_sweep_record, and on neighbour tables, it runs one pass. */
int hb_measure(hb_ctx* ctx, double M[3], double* E);

/* n_sweeps sweeps with a measurement after each, results kept on the device until the end:
 * M_series[3*s .. 3*s+2], E_series[s] (host, n_sweeps entries).  One synchronisation. */
int hb_sweep_series(hb_ctx* ctx, float T, int64_t n_sweeps, double* M_series, double* E_series);

/* Diagnostic: ONE sweep that also records every decision; accept[i] = 1 if the attempt at
 * canonical site i was accepted (host, n bytes).  Same arithmetic as hb_sweep.  Synchronises. */
int hb_sweep_record(hb_ctx* ctx, float T, uint8_t* accept);

/* Replicas (hb_lattice.n_replicas = R > 1): hb_init_*, hb_sweep, hb_sweep_count act on all replicas (hb_sweep at
 * one temperature); the calls below give every replica its own temperature and return all measurements.
 * T: R temperatures (host).  M: 3 doubles per replica; E: one per replica; series: replica-major, M_series[(r *
 * n_sweeps + s) * 3 ..], E_series[r * n_sweeps + s].  One launch per call (per 1024 sweeps of a series): replica r
 * runs in thread block r with everything resident in its SM.  hb_select_replica picks the replica that
 * hb_get_spins / hb_set_spins / hb_measure address (default 0); hb_sweep_series and hb_sweep_record need R = 1. */
int hb_sweep_each(hb_ctx* ctx, const float* T, int64_t n_sweeps);
int hb_measure_each(hb_ctx* ctx, double* M, double* E);
int hb_sweep_series_each(hb_ctx* ctx, const float* T, int64_t n_sweeps, double* M_series, double* E_series);
int hb_select_replica(hb_ctx* ctx, int32_t replica);

/* Checkpoint: (spins, sweep counter, seed, parameters) reproduce the trajectory bit for bit. */
int hb_sweep_count(hb_ctx* ctx, uint64_t* out);
int hb_set_sweep_count(hb_ctx* ctx, uint64_t value);

/* The colouring in use (host, n entries) and the number of colours.  colour may be NULL. */
int hb_get_colouring(hb_ctx* ctx, int32_t* colour, int32_t* n_colours);

/* Acceptance statistics of rule (iii) (a move is accepted if dH <= 0 or P <= exp(-beta dH)):
 * `accepts` of `attempts` moves were accepted, summed since hb_create over the COUNTED sweeps.  Counting is part of the
 * measuring colour passes (a warp vote and one atomic per warp), so the plain passes carry none of it: counted are the
 * last sweep of every hb_sweep / hb_sweep_each call, every sweep of hb_sweep_series(_each) and every hb_sweep_record
 * sweep (all replicas together).  Slab passes are not counted.  Synchronises. */
int hb_stats(hb_ctx* ctx, uint64_t* attempts, uint64_t* accepts);

/* ---- slab contexts (hb_lattice.slab_Lz > 0): one sweep of the whole lattice is, on every slab,
 *        for colour in 0 .. colours-1:  hb_slab_pass(colour);  exchange the faces of that colour with both z-neighbours;
 *        hb_slab_next_sweep()
 * Colour = (x + y + z) mod 2 in GLOBAL coordinates (sc), the basis index (bcc: 2, fcc: 4 colours; a face is then one cell
 * plane of that sublattice).  hb_slab_pass launches the colour kernel on the slab (asynchronous, on
 * the context's stream).  hb_slab_face gives, as offsets in floats into the spins buffer (hb_buffers.spins, or the
 * library's own allocation) and a length in floats, the three contiguous component runs of one face of one colour:
 * side 0 = low z, 1 = high z; ghost 0 = the slab's own boundary plane (to send), 1 = the ghost plane beyond it (to
 * receive into: the neighbour's boundary plane of the same colour).  The copy itself (cudaMemcpyPeer, NCCL send/recv,
 * peer stores) is the caller's, in stream order with the passes.  After hb_init_* / hb_set_spins the ghost planes of
 * BOTH colours must be exchanged once.  hb_measure on a slab returns its share: M = (sum over the slab's own sites) / (Lx Ly
 * slab_Lz) and the energy of its own sites with every bond counted half at each end, so that the sum over the slabs is M
 * and E of the whole lattice.  hb_get_spins / hb_set_spins move the slab's own Lx Ly Lz sites in canonical order
 * (z slowest).  hb_sweep, hb_sweep_series, hb_sweep_record and replicas return HB_ESTATE / HB_EINVAL on a slab. */
int hb_slab_pass(hb_ctx* ctx, float T, int32_t colour);
int hb_slab_next_sweep(hb_ctx* ctx);
int hb_slab_face(hb_ctx* ctx, int32_t colour, int32_t side, int32_t ghost, size_t offset_floats[3], size_t* count_floats);
/* Peer stores instead of the exchange step: after hb_slab_set_peer(ctx, side, peer_spins, peer_Lz) every colour pass of
 * this slab stores the spins it updates on its low (side 0) / high (side 1) boundary plane also into the ghost plane of
 * the z-neighbour on that side -- peer_spins is the DEVICE address, valid on this context's device, of that neighbour's
 * spins buffer (the same device, a peer device with access enabled, or an address opened from a CUDA IPC handle) and
 * peer_Lz its number of own planes (same Lx, Ly).  The transfer then overlaps the pass, store by store; what remains
 * between two passes is a barrier: no slab may start the next colour before its neighbours have finished this one
 * (stream order on one device; a collective or an event between devices).  The ghost planes must still be filled once
 * with hb_slab_face copies after hb_init_* / hb_set_spins.  peer_spins = NULL switches the side back to copies. */
int hb_slab_set_peer(hb_ctx* ctx, int32_t side, void* peer_spins, int32_t peer_Lz);
/* hb_set_option(ctx, "slab_flags", 1) (hb_diag.h; after hb_slab_set_peer on both sides; warp-specialised kernel) replaces that barrier by
 * flags between neighbours, kept in the two words behind each slab's spins (so that a peer mapping of the spins buffer
 * reaches them; hb_sizes counts them): colour pass number s of a slab takes its two boundary chunks first; a boundary tile
 * waits (acquire at system scope) until the neighbour on its side has finished the boundary chunk of ITS pass s - 1, and the
 * last warp of a boundary chunk writes s into that neighbour's flag (release at system scope) after the chunk's stores,
 * the ones into the neighbour's ghost plane included.  Interior tiles never wait.  All slabs must issue the same sequence
 * of hb_slab_pass calls, and the kernels of neighbouring slabs must be able to run at the same time (one GPU each) or in
 * the order of the passes (one stream): two processes that share one GPU must not use it.
 * With flags on, a pass is ordered only against the neighbours' NEXT pass: after the LAST pass of a run nothing on this
 * slab's stream waits for the stores the neighbours' last pass makes into its ghost planes.  Before hb_measure (boundary
 * bonds read the ghost planes), hb_get_spins on the ghost planes or hb_slab_face copies, the caller must synchronise with
 * both neighbours once (a barrier across the slabs, as without flags); DistSlab.sweep does so at the end of every call. */
/* Parts of a neighbour table (hb_lattice.part_n_total > 0; any HB_CSR context): the exchange step after a colour pass moves the
 * spins of listed sites.  hb_part_gather packs the spins of the `count` local sites ids[k] (DEVICE array of local ids) into
 * out[4 k .. 4 k + 3] = (x, y, z, 0) (DEVICE, 16-byte aligned); hb_part_scatter stores in[4 k .. 4 k + 2] as the spin of local
 * site ids[k] (ghost sites on the receiving part).  Both are asynchronous on the context's stream; the copy between the two
 * (device to device, NCCL send / recv) is the caller's.  ids out of range are an error of the caller (not checked on the
 * device); count = 0 is a no-op. */
int hb_part_gather(hb_ctx* ctx, const int32_t* ids, int64_t count, float* out);
int hb_part_scatter(hb_ctx* ctx, const int32_t* ids, int64_t count, const float* in);

/* Device memory that another process can map (one process per GPU, peer stores between slabs): hb_device_alloc is a
 * plain cudaMalloc on the current device (the result can be handed to hb_create in hb_buffers.spins), hb_ipc_export fills
 * a 64-byte CUDA IPC handle for it, hb_ipc_open maps such a handle from another process into this one and returns the
 * address to pass to hb_slab_set_peer (peer access between the two devices is enabled by the mapping), hb_ipc_close
 * unmaps.  Memory of a caching allocator (torch) cannot be exported reliably, hence the allocator here. */
int hb_device_alloc(size_t bytes, void** ptr);
int hb_device_free(void* ptr);
int hb_ipc_export(void* ptr, unsigned char handle[64]);
int hb_ipc_open(const unsigned char handle[64], void** ptr);
int hb_ipc_close(void* ptr);

/* Host-side lattice builder for a sphere cut from fcc with a free surface (A10-A12):
 * doubled integer coordinates X+Y+Z even, X^2+Y^2+Z^2 <= (2R)^2, site order ascending (Z,Y,X).
 * Core sites (12 neighbours): K_core along e_core; surface sites: K_surf along the radial direction.
 * colouring: 0 = greedy first-fit in site order, 1 = the four parity classes (X mod 2, Y mod 2).
 * Fills *out with malloc'ed tables; release with hb_lattice_free.  xyz (optional, may be NULL):
 * receives a malloc'ed 3n array of the doubled coordinates, to be free()d by the caller. */
int hb_lattice_fcc_sphere(int32_t R, float K_core, const float e_core[3], float K_surf, int32_t colouring,
                          hb_lattice* out, int32_t** xyz);
int hb_lattice_free(hb_lattice* lat);

const char* hb_strerror(int status);
const char* hb_error_detail(hb_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* HB_H_ */
