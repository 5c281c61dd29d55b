/*
 * fasttg_diag.h -- diagnostics exported by libfasttg.so that are NOT part of the library's boundary (include/fasttg.h):
 * bench.py uses them to measure the roof the attention kernels sit against.  Same conventions as fasttg.h.
 */
#ifndef FASTTG_DIAG_H_
#define FASTTG_DIAG_H_

#include "fasttg.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Times `iters` launches of a pure row-gather kernel (every group of 8
 * lanes reads 256-byte rows at pseudo-random indices of `table` [table_rows, 256 bytes] DEVICE, the access shape
 * of the attention kernels) and returns the milliseconds and the bytes gathered (HOST outputs).  With a small
 * table every access hits L1: bytes / ms is the L1 gather roof quoted in DESIGN.md section 7.  `sink`: 4 DEVICE
 * bytes.  Synchronises the stream. */
TG_API tg_status_t tg_probe_gather(const void* table, int table_rows, int gathers_per_group, int iters, void* sink,
                                   tg_stream_t stream, float* ms /*HOST*/, double* bytes /*HOST*/);
/* The same gather with an asynchronous landing zone: every group's elected lane issues one cp.async.bulk (256 bytes, completion
 * on an mbarrier) per row into a per-warp ring of `stages` (2, 4 or 8) shared-memory stages of 4 rows; the warp consumes a stage
 * with two LDS.128 per lane.  Same table, index stream and byte accounting as tg_probe_gather; `sink`: 8 DEVICE bytes;
 * *ctas_per_sm (HOST) = resident CTAs of 256 threads the ring's shared memory allowed (<= 8).  TG_ERR_INTERNAL if a copy never
 * completed (the waits are bounded).  Synchronises the stream. */
TG_API tg_status_t tg_probe_gather_bulk(const void* table, int table_rows, int gathers_per_group, int stages, int iters, void* sink,
                                        tg_stream_t stream, float* ms /*HOST*/, double* bytes /*HOST*/, int* ctas_per_sm /*HOST*/);

#ifdef __cplusplus
}
#endif
#endif /* FASTTG_DIAG_H_ */
