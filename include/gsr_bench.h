/*
 * gsr_bench.h -- measurement hook of libgsr.so, kept apart from the product ABI (gsr.h).
 * Used by bench.py for the per-kernel roofline figures; nothing in the
 * solver path calls it.
 */
#ifndef GSR_BENCH_H
#define GSR_BENCH_H

#include "gsr.h"

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    GSR_TIME_APROD1_GROUP = 1,  /* everything gsr_aprod1 launches (pack, k_aprod1, constraints)        */
    GSR_TIME_APROD2_GROUP = 2,  /* everything gsr_aprod2 launches (pre-scale, attitude kernel, main
                                   kernel, fix-up, constraints)                                         */
    GSR_TIME_K_APROD1 = 11,     /* k_aprod1 alone                                                       */
    GSR_TIME_K_APROD2_MAIN = 12,/* k_aprod2 (astro / instr / gamma scatter) alone                       */
    GSR_TIME_K_APROD2_ATT = 13, /* k_aprod2_att alone (GSR_ESTATE without the attitude copy)            */
    GSR_TIME_K_INS_SCATTER = 14,/* k_ins_scatter alone (GSR_ESTATE without the instrument copy)         */
    GSR_TIME_K_U_TO_TIME = 15,  /* k_u_to_time alone (GSR_ESTATE when u is not kept in block-time order) */
    GSR_TIME_OVERLAP_PROBE = 31,/* probe: the fused pass on one stream, k_u_to_time + k_aprod2_att on a second one,
                                   no dependency between them (time per repetition of the three).  The two
                                   streams write the handle's u / v work vectors concurrently: their contents
                                   are undefined afterwards (the next gsr_lsqr initialises them anyway)     */
    GSR_TIME_K_FUSED = 21       /* the fused pass of gsr_lsqr alone: aprod1 + the astro/instr/gamma
                                   scatter of aprod2 on one read of A (GSR_ESTATE if not in use)        */
} gsr_time_which;

/* Runs `reps` back-to-back launches of the chosen kernel(s) with the LSQR coefficients set to 0.5
 * (bounded operands) on the handle's internal u / v work vectors, after one warm-up launch, and
 * returns the mean device time per launch in milliseconds (CUDA events on the handle's stream). */
int32_t gsr_time_aprod(gsr_handle *h, int32_t which, int32_t reps, double *ms_per_launch);

/* Launch-configuration knobs for sweeps (the defaults are what gsr_create chose; DESIGN.md 5 lists the
 * sweeps they were taken from).  key: "ins_sm_fused" (instrument columns of the shared-memory accumulator
 * table of the fused pass), "n_rep" (replicas of the instrument accumulators),
 * "att_ctas_per_sm" (grid of k_aprod2_att, 1..16), "ut_ctas_per_sm" (grid of k_u_to_time, 1..16), "use_ut" (0: the fused
 * iteration gathers u through permT instead of keeping the block-time-ordered copy; 1: back, only if the handle has it),
 * "fused_nopriv" (1: fused pass without the shared-memory instrument table, REDs only; a rejected variant kept for the
 * record in DESIGN.md 5), "l2_persist" (experiment: 1 = persisting L2 access-policy window over the packed attitude
 * unknowns the fused pass gathers, 2 = over the instrument replicas its atomics hit, 0 = off and persisting lines reset).
 * "n_rep" takes 1..128 and grows the replica buffer (cudaMalloc) when the value exceeds what
 * gsr_create allocated for the product path.  GSR_EINVAL for an unknown key or a value out of range.  The captured
 * iteration is rebuilt by the next gsr_lsqr. */
int32_t gsr_bench_set(gsr_handle *h, const char *key, int64_t value);

#ifdef __cplusplus
}
#endif
#endif /* GSR_BENCH_H */
