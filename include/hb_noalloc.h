/* hb_noalloc.h -- one measurement call of libhb.so that never allocates memory.
 *
 * Who this is for.  Everything else in the library gets its working memory either from cudaMalloc or from
 * buffers the caller sized with hb_sizes() and allocated itself.  Some programs can do neither at the moment
 * they want a measurement:
 *   - a process whose device memory has been handed, all of it, to one pool (an inference server, a framework's
 *     caching allocator with a hard cap): a cudaMalloc from a guest library fails there, or eats into a budget
 *     it was never given;
 *   - a step inside a timing-critical loop: cudaMalloc and cudaFree stall the whole device until running work
 *     has drained, so a library that allocates behind the caller's back adds a hiccup the caller cannot see;
 *   - plug-in code that is given pointers to its inputs and outputs and nothing else -- no allocator handle,
 *     no place to keep a context alive between calls.
 * For these, hb_measure_sc_noalloc() computes the magnetisation M (eq. 2) and the total
 * energy E (eq. 1) of a periodic simple cubic lattice straight from three device arrays,
 * with no hb_ctx.  The block partial sums of its two-step reduction -- what hb_measure keeps in the context's
 * workspace -- live in an array that is compiled into the library image (a file-scope `static __device__`
 * array in csrc/hb_noalloc.cu).
 *
 * The price, and the limit.  That array is HB_NOALLOC_SCRATCH_BYTES = 256 KiB.  Every GPU on which the
 * library's kernels are loaded carries it from that moment until the process exits, used or not.  It has room
 * for the partial sums of HB_NOALLOC_MAX_SITES = 2^25 = 33,554,432 sites (a 322^3 lattice fits, 324^3 does
 * not); a larger lattice is refused with HB_EINVAL and a message, never truncated.
 */
#ifndef HB_NOALLOC_H_
#define HB_NOALLOC_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define HB_NOALLOC_SITES_PER_BLOCK 4096                         /* one thread block sums this many sites      */
#define HB_NOALLOC_MAX_BLOCKS 8192                              /* partial sums the static array has room for */
#define HB_NOALLOC_MAX_SITES ((int64_t)HB_NOALLOC_SITES_PER_BLOCK * HB_NOALLOC_MAX_BLOCKS)   /* 33,554,432   */
#define HB_NOALLOC_SCRATCH_BYTES (HB_NOALLOC_MAX_BLOCKS * 4 * 8)                             /* 262,144      */

/* M and E of a periodic simple cubic lattice of Lx x Ly x Lz unit spins, without a context and without
 * allocating.
 *
 * Inputs
 *   sx, sy, sz  DEVICE pointers (current device), Lx*Ly*Lz floats each: the spin components in the canonical
 *               site order of hb.h, id = (z*Ly + y)*Lx + x -- what hb_get_spins returns, copied to the device.
 *               Read only.  A host pointer here is not detected: the kernel faults, or reads whatever the GPU
 *               finds at that address.
 *   Lx, Ly, Lz  >= 1 each (periodic in all three; odd sizes are fine here, only the colour sweeps need even
 *               ones), Lx*Ly*Lz <= HB_NOALLOC_MAX_SITES.
 *   J, K, e     exchange, uniform anisotropy constant and axis (HOST pointer to 3 floats, a unit vector to
 *               1e-5 in |e|^2), as in hb_create.
 *   cuda_stream cudaStream_t the two kernels are enqueued on; NULL = the legacy default stream.
 * Output
 *   out         DEVICE pointer to 4 doubles, written in stream order: out[0..2] = M = (1/N) sum_i S_i,
 *               out[3] = E = sum_i [ -0.5 J S_i.h_i - K (S_i.e)^2 ], h_i = the sum of the six neighbours in the
 *               order -x,+x,-y,+y,-z,+z.  The arithmetic is hb_measure's: fp32 per-site terms, fp64 sums.
 *               Only the order of the fp64 additions differs, so the two agree to rounding (the test holds
 *               them to |dM| <= 1e-7 and |dE| <= 1e-6 N, the bars the parity tests use), not bit for bit.
 *               The call does not synchronise; read `out` after the stream has.
 *   err         optional HOST buffer of err_len bytes: on failure it receives a zero-terminated sentence that
 *               says what was wrong (the size limit and the size asked for, or the CUDA error text).  May be
 *               NULL.
 * Returns HB_OK, HB_EINVAL (a NULL pointer, a size < 1, more than HB_NOALLOC_MAX_SITES sites, bad J / K / e) or
 * HB_ECUDA (the address look-up or a launch failed).  After HB_EINVAL nothing has been launched.
 *
 * What the call does on the host: argument checks, at most one cudaGetSymbolAddress, two kernel launches.  It
 * never calls cudaMalloc, cudaFree, or anything else that allocates, and it keeps no per-call state.
 *
 * First call on each device.  The address of the static array differs from GPU to GPU, and host code cannot
 * take it with `&`; the first call made while a given device is current asks the runtime for it
 * (cudaGetSymbolAddress) and remembers the answer for that device.  That look-up may make the runtime load the
 * library's kernels onto the device.  Make this first call during start-up, with the device you will use
 * current (cudaSetDevice), and before any stream capture begins.  Later calls only launch.
 *
 * Sharing.  There is ONE array per GPU, and every call on that GPU uses it.  The first kernel overwrites each
 * partial sum the second one will read, so nothing has to be zero beforehand and whatever an earlier call left
 * behind is harmless.  But two calls that run on the GPU at the same time -- different streams, or different
 * host threads on different streams -- write the same words and give wrong sums: put all calls for one GPU on
 * one stream, or order them with events.  Calls on different GPUs do not interfere.
 */
int hb_measure_sc_noalloc(const float* sx, const float* sy, const float* sz, int32_t Lx, int32_t Ly, int32_t Lz,
                          float J, float K, const float e[3], double* out, void* cuda_stream,
                          char* err, size_t err_len);

#ifdef __cplusplus
}
#endif
#endif /* HB_NOALLOC_H_ */
