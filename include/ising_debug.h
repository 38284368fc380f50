/*
 * ising_debug.h -- diagnostics of the B200-native Ising annealer.  NOT part of the product boundary (include/ising.h):
 * nothing here changes a result; it only records where the persistent Gauss-Seidel kernel spends its time.
 */
#ifndef ISING_B200_DEBUG_H
#define ISING_B200_DEBUG_H

#include "ising.h"

#ifdef __cplusplus
extern "C" {
#endif

/*
 * The next ising_anneal calls (persistent cooperative-grid Gauss-Seidel kernel only) record, for sweep `sweep` of the
 * call, the SM clock of every CTA when it arrives at and when it leaves the grid barrier that ends each virtual phase
 * (the colour phases; with a tail chain: the phases before the tail, the bulk pseudo-phase, then the chain).
 *   stamps   uint64 [ising_problem_info(15) + 1][ising_problem_info(12)][8], DEVICE: word 0 arrival, word 1 departure,
 *            words 2-7 unused; NULL switches the recording off
 * Stamps of different CTAs come from different SM clocks: compare differences within one CTA.
 */
ising_status ising_debug_phase_timing(ising_problem* p, uint64_t* stamps, int32_t sweep);

/*
 * Bandwidth probe (measurement only): what this GPU's L2 sustains for the access patterns of the sparse sweep.
 *   scratch        DEVICE memory, at least `bytes` long (a power of two >= 1 MiB is used: the largest that fits)
 *   gather_gbs     HOST out: random 32-byte sector gathers from the buffer, GB/s of sectors delivered: the better of two
 *                  access shapes (two 16-byte loads per lane pair = 16 sectors per warp instruction, the sweep's shape;
 *                  4-byte loads by eight lanes per sector = 4 sectors per instruction), eight loads in flight per lane
 *   gather16_gbs   HOST out: the same for the 16-byte shape alone (what the sweep kernel's gathers can reach)
 *   stream_gbs     HOST out: grid-strided 16-byte streaming reads of the same buffer, GB/s
 * Pick `bytes` = the state size of interest (config 5: 32 MiB, L2-resident).  Synchronises `stream`.
 */
ising_status ising_debug_probe_l2(void* scratch, size_t bytes, double* gather_gbs, double* gather16_gbs, double* stream_gbs,
                                  void* stream);

#ifdef __cplusplus
}
#endif
#endif /* ISING_B200_DEBUG_H */
