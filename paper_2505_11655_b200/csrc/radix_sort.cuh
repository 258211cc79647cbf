// Device-resident LSD radix sort (8-bit digits) of uint64 keys with an optional uint32 payload.
// Used by the sky sort of the fused lnL path (keys = delay cells, payload = sample index) and
// by the AV cell-set build (keys only).  Both the element count and the number of significant
// key bits live in device memory, so a sort can follow a device-side decision (N_min, n_bins)
// with no host round-trip: passes above the significant bits exit immediately.
#pragma once
#include "common.cuh"

#define RS_TILE 4096          // keys per block (8 warps x 16 rounds x 32 lanes)
#define RS_THREADS 256
#define RS_MAX_PASSES 8

struct RadixSortPlan {
    int max_n;                // capacity the buffers were sized for
    int max_blocks;           // ceil(max_n / RS_TILE)
    uint32_t* hist;           // [256][max_blocks] per pass (reused), digit-major, + 256 row totals
    size_t bytes;             // scratch bytes behind hist
};

// scratch the caller must provide for capacity max_n (bytes)
size_t radix_sort_scratch_bytes(int max_n);

// Sorts keys (and vals) ascending, stable.  n_dev: device int64 element count (<= max_n);
// bits_dev: device int, number of significant low key bits (<= 64; passes = ceil(bits/8)).
// Ping-pongs between (k0, v0) and (k1, v1); the result is in buffer (passes & 1): the caller
// reads it through radix_sort_result_kernel-style indirection, or calls radix_sort_finish to
// copy it back into (k0, v0) when passes is odd.  v0/v1 may be NULL (keys only).
int radix_sort_device(ile_ctx* ctx, int max_n, const long long* n_dev, const int* bits_dev, uint64_t* k0, uint32_t* v0,
                      uint64_t* k1, uint32_t* v1, void* scratch, int max_passes);
