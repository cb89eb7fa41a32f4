/*
 * ajt_test.h — test hooks and measurement helpers of libajt.so.  Not part of the method (include/ajt.h is the
 * product's C ABI); tests/ and bench.py use these.
 */
#ifndef AJT_TEST_H_
#define AJT_TEST_H_

#include "ajt.h"

#ifdef __cplusplus
extern "C" {
#endif

/* ajt_merge_timelines / ajt_merge_blocks `flags` */
enum {
    AJT_MERGE_WEAK_HASH = 1 /* degrade the prefix hash to 4 bits so that hash-equal, token-different
                               candidates are common and the exact comparison that guards every accepted
                               candidate is exercised.  Results are still exact (AJT_STATUS_HASH_COLLISION is set). */
};

/* Measurement helper ("a micro-benchmark for read-only, write-only and copy HBM ceilings on the same box"):
 * streams `bytes` (multiple of 16, 16-byte aligned DEVICE buffers) with 16-byte accesses.  mode 0: read `src` (dst = a DEVICE
 * word that is practically never written, may alias anything), 1: write zeros to `dst`, 2: copy src -> dst, 3: cudaMemsetAsync
 * of `dst`. */
int ajt_hbm_probe(void* dst, const void* src, size_t bytes, int32_t mode, ajt_stream_t stream);

/* Kernels launched by the library in this process so far (every launch site counts itself).  bench.py reads it on both
 * sides of the timed region to report `gpu_launches`. */
uint64_t ajt_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif /* AJT_TEST_H_ */
