// measure_api.h -- C entry points that exist ONLY in the measurement library
// (libculgt_b200_measure.so, python -m paper_1412_3655_b200.build --measure).  Not part of the
// product ABI (include/culgt_b200.h).
#pragma once
#ifdef CULGT_MEASURE
#include "../../include/culgt_b200.h"
#ifdef __cplusplus
extern "C" {
#endif
/* culgt_or_sweeps with a workspace (>= culgt_workspace_bytes, used exclusively by this call while it
 * runs): variant 60 runs every sweep as the fused one-kernel schedule of or_sweep_fused.cu; the
 * result is bit-identical to culgt_or_sweeps. */
int culgt_or_sweeps_ws(const culgt_lattice* lat, void* links, void* workspace, int n_sweeps, double omega,
                       void* stream);
/* Host-only: the order in which the fused full sweep hands out its 2*n_slices slice-tasks,
 * tasks_out[u] = parity << 31 | time-slice (n_slices even, 2..512; lag clamped to [1, n_slices-2];
 * direction 0 ascending, 1 descending). */
int culgt_fused_schedule(int n_slices, int lag, int direction, unsigned* tasks_out);
#ifdef __cplusplus
}
#endif
#endif
