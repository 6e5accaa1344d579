// gcm_multi.cuh -- launch interface of the many-large-messages-under-one-key kernel (gcm_multi.cu):
// config C3, FITS-sized HDUs through the batched API (include/gcm.h).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "gcm_common.cuh"

// One message of the group, device memory: the row loop's view of it (gcm_common.cuh: RowMsg, the same virtual
// block sequence [pad | AAD | payload | length block] as the single-message kernel) plus IV, expected tag and the
// slot its result goes to.
struct MultiMsg {
    RowMsg   m;
    uint32_t iv[3];
    uint32_t result;          // index into the result array
    uint32_t tag_expect[4];   // decrypt
};

// Rows [r0, r1) of message msg: the unit of work of one warp.  Warp w owns chunks
// [warp_first[w], warp_first[w + 1]).
struct MultiChunk { uint32_t msg, r0, r1, reserved; };

struct MultiResult { uint32_t tag[4]; int status; int pad[3]; };   // == BatchResult of gcm_batch.cu

struct MultiParams {
    uint32_t rk[60];
    uint32_t te0[256];        // round table T0 (see GcmParams)
    GcmTables tab;
    const MultiMsg   *msgs;
    const MultiChunk *chunks;
    const uint32_t   *warp_first;
    uint32_t n_msgs;
    uint32_t n_warps;         // warps that own at least one chunk
    unsigned long long *acc;  // per message: 2 x 64 bit GHASH accumulator, zeroed before the launch
    unsigned *counter;        // last-CTA-done ticket, zeroed before the launch
    MultiResult *results;
};

#define MULTI_THREADS 512

cudaError_t launch_multi(int nr, int mode, int blocks, const MultiParams &p, cudaStream_t s);
// zero-fills the outputs of the messages whose status is non-zero (payload suppression)
void launch_multi_wipe(const MultiMsg *msgs, const MultiResult *results, uint32_t n_msgs, cudaStream_t s);
