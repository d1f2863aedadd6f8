/* hb_diag.h -- tuning knobs and diagnostics of libhb.so, kept apart from the product calls of hb.h.
 *
 * Nothing here is needed to run the method of arXiv 2106.11286 (hb.h: hb_create, hb_sweep, hb_measure and the series /
 * replica / slab / part calls).  These entry points exist to MEASURE the library: the ceilings its rooflines are quoted
 * against (hb_probe_alu, hb_probe_pipe, hb_probe_sc_l2), the arithmetic contract element by element
 * against the CPU oracle (hb_device_math), the paper's own racy update scheme as context
 * (hb_sweep_paper_scheme), launch counters, and the kernel options that choose between variants which
 * all compute the same bits (hb_set_option).  Conventions (status codes, host / device pointers) are those of hb.h.
 */
#ifndef HB_DIAG_H_
#define HB_DIAG_H_

#include "hb.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Counters since hb_create: kernels launched by this context, sites attempted. */
int hb_counters(hb_ctx* ctx, uint64_t* kernel_launches, uint64_t* attempts);

/* Diagnostic: the rate (attempted updates per second) at which this device executes the attempt arithmetic alone --
 * Philox, proposal, neighbour sum on registers, delta-H, acceptance; no memory traffic -- in launches issued back to back on
 * `cuda_stream` for about `seconds` (0 < seconds <= 10; the second half is timed, so the clock is the one a long run
 * holds).  It is the arithmetic ceiling of the colour kernels on this chip.  Synchronises. */
int hb_probe_alu(void* cuda_stream, double seconds, double* updates_per_second);

/* Diagnostic (self-test of the arithmetic contract): evaluates on the current device, element by
 * element, the building blocks of one attempt exactly as the colour kernels evaluate them -- the scalar functions AND the
 * packed fp32x2 copies the tuned kernels use -- so that tests can compare them bit for bit with the CPU oracle over every
 * argument that can occur.  Host pointers; `count` elements (at most 2^26); synchronises; uses the legacy default stream.
 *   HB_MATH_U01     out[2i] = u(in0[i]) scalar, out[2i+1] = packed                        (u(r) = (2 (r >> 9) + 1) 2^-24)
 *   HB_MATH_SINCOS  out[2i] = sin, out[2i+1] = cos of 2 pi k / 2^24, k = (in0[i] >> 8) | 1
 *   HB_MATH_SPHERE  out[6i..6i+2] = proposal (x, y, z) from random words (in0[i], in1[i]), scalar; out[6i+3..6i+5] packed
 *   HB_MATH_EXP     out[2i] = exp_spec(x) scalar, out[2i+1] packed; x = the float whose bits are in0[i], in [-17, 0]
 *   HB_MATH_SQRT    out[2i] = the library's square root of w = 1 - (1 - 2 u(in0[i]))^2, out[2i+1] = IEEE sqrt of the same w
 *   HB_MATH_ATTEMPT one whole packed attempt per element: in0[i] = site id, in1[16i..] = (sweep_lo, sweep_hi, seed_lo,
 *                   seed_hi) as integers and (J, K, beta, ex, ey, ez, hx, hy, hz, sx, sy, sz) as float bits; elements 2t and
 *                   2t+1 form a pair and use (J, K, beta, e) of element 2t; out[4i..] = the spin after the attempt, accepted */
enum { HB_MATH_U01 = 0, HB_MATH_SINCOS = 1, HB_MATH_SPHERE = 2, HB_MATH_EXP = 3, HB_MATH_SQRT = 4, HB_MATH_ATTEMPT = 5 };
int hb_device_math(int32_t op, int64_t count, const uint32_t* in0, const uint32_t* in1, float* out);

/* Context, not the product path: n_mcs Monte Carlo steps per spin of the PAPER'S OWN update scheme (PAPER.md
 * lines 30-32), emulated: the linearised array is cut into N / n_per_block "blocks" of n_per_block consecutive sites, at
 * every step every block updates ONE randomly chosen spin of its own against whatever its neighbours hold in global memory
 * at that moment (other blocks update theirs concurrently: racy by construction, "loss of continuity" for small n), one
 * launch per step, n_per_block steps per MCS.  The paper's choice is n_per_block = 8.  Not reproducible bit for bit and
 * never compared with the trajectory oracle: only its statistics (against the fp64 random-site oracle) and its rate mean
 * anything.  Simple cubic, whole lattice.  The sweep counter advances by n_mcs; hb_stats counts every attempt.  Asynchronous. */
int hb_sweep_paper_scheme(hb_ctx* ctx, float T, int64_t n_mcs, int32_t n_per_block);

/* Diagnostic: the issue rate of one instruction kind (or mix) the colour kernels are made of, in warp-instructions per clock
 * per SM (4.0 = one per clock on each of the four sub-partitions), measured with the SM clock over a loop of 8 independent
 * register chains per thread, 32 warps per SM.  It is the measurement behind the arithmetic ceiling of DESIGN.md section 7
 * (a Philox round costs IMAD.WIDE + LOP3; packed fp32x2 costs two scalar slots).  Mixes count every named kind.
 * Synchronises. */
enum { HB_PIPE_FFMA = 0, HB_PIPE_FFMA2 = 1, HB_PIPE_IMAD = 2, HB_PIPE_IMAD_WIDE = 3, HB_PIPE_LOP3 = 4,
       HB_PIPE_WIDE_LOP3 = 5, HB_PIPE_FFMA_WIDE_LOP3 = 6, HB_PIPE_FFMA2_WIDE_LOP3 = 7 };
int hb_probe_pipe(void* cuda_stream, int32_t kind, double* warp_instr_per_clk_per_sm);

/* Diagnostic: the rate (attempted updates per second) of the warp-specialised simple cubic colour kernel when its HBM
 * traffic is taken away: n_sweeps sweeps (two launches each, timed with CUDA events after two untimed ones) in which plane z
 * is read and written at the address of plane z mod `planes` (a power of two, e.g. 16), so that the whole launch lives in
 * a few L2-resident planes while every attempt is still computed.  It is the ceiling of any scheme that keeps the kernel's
 * arithmetic and only removes DRAM traffic (fused colours, temporal blocking: DESIGN.md 6.9).  The result is NOT a
 * trajectory: the call leaves the spins undefined (HB_ESTATE until hb_init_* / hb_set_spins).  Simple cubic, whole lattice,
 * rows that fit the kernel's 7-row variant.  Synchronises. */
int hb_probe_sc_l2(hb_ctx* ctx, float T, int64_t n_sweeps, int32_t planes, double* updates_per_second);

/* Tuning knobs, by name (DESIGN.md section 6 lists them); unknown names give HB_EINVAL. */
int hb_set_option(hb_ctx* ctx, const char* name, int64_t value);
int hb_get_option(hb_ctx* ctx, const char* name, int64_t* value);

#ifdef __cplusplus
}
#endif
#endif /* HB_DIAG_H_ */
