/*
 * cs_select_batch.h -- compaction of the candidate lists of several scales in ONE cooperative launch (cs_select.cu).
 * A multi-scale handle (cfg 5, four grids) compacts its lists at the same points of the re-scan;
 * one launch each left most SMs idle (a 2^18-entry list is 128 tiles on 148 x 4 CTA slots) and paid the launch and the
 * grid barriers four times.
 */
#ifndef CS_SELECT_BATCH_H_
#define CS_SELECT_BATCH_H_

#include "cs_internal.h"

namespace cs {

struct CompactRequest {
    const SelectBuffers* B;   /* buffers of the scale (room for `cap` entries each half) */
    int src;                  /* half that holds the list */
    uint32_t n;               /* entries */
    int id_bits;              /* ids < 2^id_bits */
    ScanState* st_dev;        /* device state of the scale */
    uint32_t* epoch;          /* per-buffer sweep counter (host) */
};

/* Enqueues the compaction of `count` <= CS_MAX_SCALES lists (same cap, k_max, thr_min) on `stream`: one cooperative launch
 * for the lists that hold entries, one single-thread launch per empty list.  No synchronisation.  *launches += launches. */
cudaError_t select_compact_batch(const CompactRequest* req, int count, uint32_t cap, uint64_t k_max, int32_t thr_min,
                                 cudaStream_t stream, uint64_t* launches);

}  // namespace cs
#endif
