/* dns_debug.h -- TEST AND MEASUREMENT HOOKS of libdns_b200.  Not part of the product ABI (include/dns.h): nothing a
 * user of the time stepper needs is declared here.  tests/ and bench.py use these calls to look at per-stage internals, to
 * force the code paths the defaults do not take (so that every kernel family is parity-tested), and to measure the fp64
 * peak the roofline fractions are quoted against.  Same conventions as dns.h: int status, nothing throws. */
#ifndef DNS_B200_DEBUG_H
#define DNS_B200_DEBUG_H

#include "dns.h"

#ifdef __cplusplus
extern "C" {
#endif

/* dns_debug_fetch -- test hook: copy one INTERNAL device array to a host buffer, synchronising first.  Internal
 * spectral layout is [Ny][nkx][nkz][E] complex128 (member index fastest).  which: 0 u, 1 w, 2 du/dy, 3 dw/dy
 * (current stage, Eq. 17-18; in the rotational form 2 is omega_z = i kx v - du/dy and 3 is omega_x = dw/dy - i kz v), 4 the three spectral advection terms (u.grad)u,(u.grad)v,(u.grad)w back to back,
 * 5 F and 6 G history (Eq. 4-5, interior rows: F^0 after stage 0, F^0 + 4 F^1 after stage 1), 7 v of
 * the current stage, 8 U00 and
 * 9 W00 of the current stage as [Ny][E] float64, 10 eta of the current stage (rotational form only; stages 0 and 1).  nbytes must equal the array size (DNS_EINVAL otherwise). */
int dns_debug_fetch(dns_plan* plan, int which, void* host_dst, size_t nbytes);

/* dns_debug_stage -- test hook: enqueue ONE Crank-Nicolson/RK3 stage (0, 1 or 2) on the
 * plan's stream, so that per-stage internals can be fetched.  A step is stages 0, 1, 2 in order; the step
 * counter advances after stage 2.  Errors: DNS_EINVAL (stage outside 0..2), DNS_ESTATE, DNS_ECUDA. */
int dns_debug_stage(dns_plan* plan, int stage);

/* dns_debug_set_option -- process-wide tuning / path-selection options, read by dns_plan_create (and "graph" by
 * dns_step).  value < 0 restores the default (the measured best).  Names:
 *   "graph"    0: dns_step launches directly instead of replaying the CUDA graph of one step
 *   "zreg"     0: shared-memory z transforms instead of the register-resident ones
 *   "etf"      member tile of the shared-memory z transforms (4, 8, 16, 32)
 *   "ety","nty" member tile (4, 8, 16) and n-tiles per warp (1, 2, 4) of the per-pair kernel
 *   "line_tps" lanes per slot of the line kernel (4, 8, 16)
 *   "line_ring" input ring of the line kernel with 16-lane tiles: 0 half an item deep, 1 a whole item (8 | 6 fields)
 *   "line_pair" Mx = 54, 72 (12 slots, 6 busy in the first pass): 0 one transform per round; 1 two per round with two
 *              exchange buffers, 5 with four buffers and a half ring (both convective form only); default: two per round,
 *              four buffers, 6-slot ring
 *   "zinv_tp"  0: convective form without the L2 prefetch of the two-pass z inverse (Mz <= 48) and, for Mz = 72, with the
 *              one-pass kernel (8 output fields) instead of the two-pass one
 *   "pdl"      1: programmatic dependent launch between the stage kernels (measured slower: off by default)
 *   "line_alt" 1: Mx = 72 as 8 x 9 on 9 one-warp slots in the line kernel instead of 6 x 12 on 12 slots (measured slower)
 * Errors: DNS_EINVAL (unknown name). */
int dns_debug_set_option(const char* name, int value);

/* dns_debug_fp64_peak -- measures the sustained fp64 throughput of the current device with a register-resident
 * microbenchmark (no memory traffic): kind 0 = DFMA chains, kind 1 = DMMA.8x8x4 (mma.sync m8n8k4 f64) chains, kind 2 = both kinds
 * interleaved in every thread (8 DFMA + 2 DMMA chains: the sum stays below either peak, i.e. the two share one pipe), run back
 * to back for about `seconds` of device time; *tflops receives 2 x fused multiply-adds per second / 1e12.  This is the
 * denominator of every fp64 roofline fraction bench.py prints ("measure sustained fp64 ... exactly as
 * MEASURED_PEAKS.json did for bf16").  Errors: DNS_EINVAL, DNS_ECUDA. */
int dns_debug_fp64_peak(int kind, double seconds, double* tflops);

#ifdef __cplusplus
}
#endif
#endif /* DNS_B200_DEBUG_H */
