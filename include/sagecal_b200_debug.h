/*
 * sagecal_b200_debug.h -- host-only TEST HOOKS of libsagecal_b200.so
 *
 * Not part of the product API (include/sagecal_b200.h): these entry points replay, on the host and without a device,
 * how the kernels split their work, through the same geometry routines the launches use, so that CPU tests can check
 * that every sample / baseline / record is touched exactly once (tests/test_abi_host.py).  They compute nothing of the
 * method.
 */
#ifndef SAGECAL_B200_DEBUG_H
#define SAGECAL_B200_DEBUG_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/*
 * Test hook, host only, no device needed: replays the work decomposition of the LM pass kernel.
 * cover : host out [T*B] int32, must be zeroed by the caller; on return every entry must be 1 (each baseline and
 *         time slot visited by exactly one thread of one CTA).
 * info  : host out [8] int64 = {TQ, nchunk, ncols, TC, tlen, nslots, R, U}.
 * Returns 0, SAGECAL_EINVAL, or a positive bit mask naming the violated bookkeeping invariant.
 */
int sagecal_debug_pass_cover(int nstations, int ntime, int nchan, int32_t* cover, int64_t* info);

/*
 * Test hook, host only: replays the work decomposition of the compressed M-step kernel (one thread per
 * baseline, a warp per chunk of rows of one 32-column segment) and the record lists of its station reduction, for a
 * device with `sms` SMs, through the same geometry routines the launch uses.  cover : host out [B] int32, zeroed by the
 * caller; every entry must come back 1.  info : host out [8] int64 = {column segments, rows per chunk, chunks, B, units,
 * units visited, grid, shared-memory slots per warp}.  Returns 0, SAGECAL_EINVAL, or a positive bit mask (1/4: a
 * row/column record is read but never written; 2/8: a record that carries a baseline is never read; 16/32: a chunk or
 * record index out of range; 64: a unit visited twice).
 */
int sagecal_debug_mstep_cover(int nstations, int sms, int32_t* cover, int64_t* info);

/*
 * Test hook, host only: replays the fragment addressing of the tensor-core statistics kernel (DESIGN.md §5.5 "cluster
 * groups", 2x2 form): one warp per baseline walks its T*F samples 8 at a time; every lane touches one double of two
 * samples as C/D/A fragment and two doubles of one sample as B fragment of the write-back.
 * cover_cd, cover_b : host out [T*B*F*8] int32 each, zeroed by the caller: how often each double of each sample is
 *                     addressed in either role; every entry must come back 1 (nothing missed, nothing twice).
 * Returns 0, SAGECAL_EINVAL, or a positive bit mask (1/2: an address outside the array in either role).
 */
int sagecal_debug_mma_cover(int nstations, int ntime, int nchan, int32_t* cover_cd, int32_t* cover_b);

#ifdef __cplusplus
}
#endif

#endif /* SAGECAL_B200_DEBUG_H */
