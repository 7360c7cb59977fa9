/*
 * nhplan_probe.h -- measurement probes of libnhplan.so, NOT part of the planner's interface: two micro-benchmarks that
 * bench.py runs next to the plan to state the machine limits its roofline lines are read against (DESIGN.md sections 6, 6.7).
 * They take a planner handle only for its stream, its device and (the read probe) its value volume, and change nothing a
 * plan depends on.
 */
#ifndef NHPLAN_PROBE_H
#define NHPLAN_PROBE_H

#include "nhplan.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Integer-pipe micro-benchmark behind bench.py's `alu` line: launches a kernel of `chains`
 * (1..8) independent VIADDMNMX (add + min, the instruction every sweep step is made of) dependency chains per thread on the
 * handle's stream, 8 warps per SM sub-partition on every SM, times it with CUDA events and returns the throughput in
 * lane-operations per second (*lane_ops_per_s) and the SM count used (*sms).  Touches none of the planner's volumes.
 * Synchronises the stream.  Errors: NHP_E_ARG, NHP_E_CUDA. */
int nhp_microbench_alu(nhp_planner *p, int chains, double *lane_ops_per_s, int *sms);

/* Read probe behind the roofline discussion: reads the whole value volume V once, nothing else, in the
 * access pattern of one of the sweep kernels -- 0: linear 4 KB chunks, 1: straight_rows_kernel (a warp walks a band: 32 rows of
 * 128 bytes per tile), 2: straight_xl_kernel (tiles follow each other along the rows), 3: turn_tile_kernel (one CTA per tile of 32
 * curves, warp s reads planes 32 s .. 32 s + 31) -- on the handle's stream, timed with CUDA events, and returns bytes per second.
 * V is not modified (its content does not matter).  Synchronises the stream.  Errors: NHP_E_ARG, NHP_E_CUDA. */
int nhp_microbench_read(nhp_planner *p, int pattern, double *bytes_per_s);

#ifdef __cplusplus
}
#endif
#endif /* NHPLAN_PROBE_H */
