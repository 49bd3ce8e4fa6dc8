/* nh_debug.h -- tuning and test hooks of libnh_b200.so.  NOT part of the contract (include/nh.h is): the keys,
 * their meaning and their defaults may change with any build.  Results do not depend on any of them (the GPU tests
 * check bit-identity across them); they only move work between launch shapes that were measured against each
 * other on B200.  The value 0 always means "the library decides". */
#ifndef NH_DEBUG_H
#define NH_DEBUG_H
#include "nh.h"
#ifdef __cplusplus
extern "C" {
#endif

#define NH_TUNE_FD_PLANES        0   /* planes per CTA of the tiled FD kernels                                      */
#define NH_TUNE_LB2_LEAD         1   /* two-step LB kernel: lead D of phase 1 over phase 2, in planes               */
#define NH_TUNE_LB2_RING         2   /* two-step LB kernel: ring planes R (>= D + 2)                                */
#define NH_TUNE_LB2_STRIPS       3   /* two-step LB kernel: number of y-strips (must divide ny; <= 32)              */
#define NH_TUNE_LB2_CELLS        4   /* two-step LB kernel: cells per thread (1, 2 or 4)                            */
#define NH_TUNE_LB2_THREADS      5   /* two-step LB kernel: threads per CTA, 64 ... 256 in steps of 32 (where they tile) */
#define NH_TUNE_LB2_BLOCKORDER   6   /* two-step LB kernel: units in blockIdx order instead of by atomic ticket;
                                        relies on in-order CTA dispatch, which CUDA does not promise: tuning only,
                                        a violated order ends in the wait's timeout (NH_ECUDA), not in a hang       */
#define NH_TUNE_LB2_TIMEOUT_MS   7   /* two-step LB kernel: bound of one dependency wait (default about 4000 ms)    */
#define NH_TUNE_LB2_FAULT        8   /* test hook: the waits of the next launches ask for an epoch that never comes,
                                        so they time out and the lattice reports NH_ECUDA from then on             */
#define NH_TUNE_COUNT            9

/* Set one knob.  Synchronises the lattice's stream if graphs were captured (they are dropped).  NH_EINVAL for a
 * null handle, an unknown key or a negative value. */
int nh_debug_tune(nh_lattice* L, int key, int value);

#ifdef __cplusplus
}
#endif
#endif
