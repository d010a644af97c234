/*
 * u1u1_tuning.h -- experimental switches of libu1u1.so.  NOT part of the supported boundary (include/u1u1.h): they
 * select staging paths, grid orders, cache policies and chunk lengths that were measured while the kernels were
 * written and exist so that tests can prove the alternatives bit-identical.  Production code
 * leaves them at 0.  Every combination computes the same step (Eq. 17-26) and the same diagnostics.
 */
#ifndef U1U1_TUNING_H
#define U1U1_TUNING_H

#include "u1u1.h"

#ifdef __cplusplus
extern "C" {
#endif

#define U1U1_TUNE_SCALAR_CHAIN 1u    /* variant 0 in scalar instead of packed fp32x2 instructions (same bits); one-step kernel */
#define U1U1_TUNE_NO_TMA 2u          /* cp.async staging everywhere (step kernels and diagnostics sweep)          */
#define U1U1_TUNE_MOM_LDCS 4u        /* one-step kernel: momenta by ld.global.cs                                */
#define U1U1_TUNE_PLAIN_GRID 8u      /* one-step kernel: plain grid order                                        */
#define U1U1_TUNE_DIAG_L2_A 16u      /* diagnostics sweep: L2 policies                                           */
#define U1U1_TUNE_DIAG_L2_B 32u
#define U1U1_TUNE_DIAG_CHUNK16 64u   /* diagnostics sweep: 16 / 32-plane chunks                                  */
#define U1U1_TUNE_DIAG_CHUNK32 128u
#define U1U1_TUNE_ONE_STEP 256u      /* one-step kernel even with an aux buffer                                  */
#define U1U1_TUNE_TB_CHUNK16 512u    /* two-step kernel: 16 / 64-plane chunks                                    */
#define U1U1_TUNE_TB_CHUNK64 1024u
/* 2048 is taken: it is what u1u1_params.range_reduce turns on */
#define U1U1_TUNE_ALL 2047u

/* Replace the context's experimental switches (a mask of U1U1_TUNE_*; bits outside U1U1_TUNE_ALL -> U1U1_EINVAL).
 * Takes effect at the next launch; survives configure / set_params. */
int u1u1_set_tuning(u1u1_ctx *ctx, uint32_t flags);

#ifdef __cplusplus
}
#endif
#endif /* U1U1_TUNING_H */
