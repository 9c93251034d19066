// dev_consts.h -- constants and bit layouts shared by host code, the statically compiled kernels and
// the run-time specialised (NVRTC) chunk kernels.  Macros only: no includes, no types.
#pragma once
#define SG_NMAX 32     /* table size: SMOLGP_MAX_DIM (31) + 1; the chunk kernels give each of the n + 1 columns a lane */
#define SG_MAXINST 16  /* max number of instruments (= SMOLGP_MAX_INST) */
#define SG_MAXBLK 16   /* max number of block-diagonal blocks of F (App. C.1 stacking) */
#define SG_MAXBD 4     /* max block dimension */
#define SG_DENSE_NT 256 /* threads of the CTA that works on one dense combine */
#define NUMF_BAD 1     /* numeric flag: non-finite value or non-positive innovation variance */
#define NUMF_SIGMA 2   /* noise_sigma <= 0 or not finite at an exposure */
#define NUMF_AMP 4     /* amp <= 0 or not finite for a series */

// event meta word: bit 0 kind (1 = start/reset, 0 = end/observe), bits 1..5 instrument,
// bits 8..23 zero-mask Z_k (instruments whose z is zeroed after event k: idle ones, and the
// event's own instrument in both cases: reset at a start, idle after an end).
#define META_KIND(m) ((m) & 1u)
#define META_INST(m) (((m) >> 1) & 31u)
#define META_ZMASK(m) (((m) >> 8) & 0xFFFFu)
