/*
 * hadpsgd_oracle.h -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, single-threaded CPU definition of one H-ADPSGD super-learner
 * step, written from /root/reference/PAPER.md (arxiv 1907.05701) and the
 * readings listed in DESIGN.md section 3.  It shares no code, header, table or
 * helper with the CUDA path under paper_1907_05701_b200/.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may load it.
 *
 * Every function here is pinned by tests/test_oracle_pins.py against closed
 * forms, exact-rational arithmetic, brute-force dense mixing matrices and the
 * invariants the paper states; no function is "parity unpinned".
 *
 * All pointers are HOST pointers.  Layout is row-major:
 *     grads[s][g][i]  (S*G*P elements; fp32, or bf16 stored as uint16)
 *     w[s][i], v[s][i] (S*P fp32, or S*P fp64 for the _f64 shadow)
 * Return value: 0 = ok, -1 = invalid argument.
 */
#ifndef HADPSGD_ORACLE_H
#define HADPSGD_ORACLE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum { ORACLE_GRAD_F32 = 0, ORACLE_GRAD_BF16 = 1 };

/* flags */
enum {
    ORACLE_NO_MIX       = 1u << 0, /* T_k = I : every super-learner keeps u_s (eq. (6)/(3) only)     */
    ORACLE_EQ7_LITERAL  = 1u << 1  /* eq. (7) as printed: w'_s = 1/2 (w_s + w_p) - lr * v_s           */
};

/* Pairing (reading R7; "left or right neighbor in the
 * ring"): even step_k pairs (2i, 2i+1); odd step_k pairs (2i+1, (2i+2) mod S).
 * S == 1 -> partner[0] = 0.  S odd and > 1 -> -1 (no perfect matching, R8).   */
int hadpsgd_oracle_partner(int S, uint64_t step_k, int32_t* partner /*[S]*/);

/* Dense mixing matrix T_k (symmetric, doubly stochastic, two 0.5
 * per row and column).  With the update-then-average reading (R3) a pair
 * (s,p) contributes T[s][s]=T[s][p]=T[p][s]=T[p][p]=0.5.  Row-major S x S.   */
int hadpsgd_oracle_mixing_matrix(int S, uint64_t step_k, double* T /*[S*S]*/);

/* One step, fp32 storage and fp32 arithmetic, one rounding per operation, no
 * FMA contraction (compiled -ffp-contract=off), fixed left-to-right learner
 * order.  This is the bit pattern the CUDA path must reproduce in its
 * deterministic mode.
 *   phase 1 (eq. (6) PAPER.md:57 then eq. (3) PAPER.md:34 + momentum, R2):
 *       acc  = grads[s][0][i] + grads[s][1][i] + ... (left to right)
 *       gbar = acc * (1.0f/G)
 *       v    = mu*v + gbar          (mul, then add)
 *       u    = w - lr*v             (mul, then sub)
 *   phase 2 (eq. (7), T_k PAPER.md:66, order per PAPER.md:62, R3):
 *       w_s = w_p = 0.5f * (u_s + u_p)
 *   with ORACLE_EQ7_LITERAL (eq. (7) as printed; fp32 order fixed by R14):
 *       m = 0.5f * (w_s + w_p)  (OLD weights) ;  t_s = lr * v_s  (the new v) ;  w_s = m - t_s
 * diag (optional, may be NULL): doubles laid out  (R14)
 *       gsq[S] | wsq[S] | gap[S]   (gap[s] == gap[partner[s]]; exactly 0 if unpaired)
 *   gsq[s] = sum_i gbar^2, wsq[s] = sum_i w'_s^2 (the weights s holds after the step),
 *   gap[s] = sum_i (a_s-a_p)^2 over the two vectors the mix averages: a = u by default,
 *   a = the OLD weights w under ORACLE_EQ7_LITERAL; each term formed in double from the
 *   fp32 values.
 * grads are read-only; w and v are updated in place.                          */
int hadpsgd_oracle_step(int S, int G, int64_t P,
                        const void* grads, int grad_dtype,
                        float* w, float* v,
                        float lr, float mu, uint64_t step_k, uint32_t flags,
                        double* diag /* [3*S] or NULL */);

/* The same step for a CALLER-SUPPLIED matching (R8): partner
 * [S] must be an involution (partner[partner[s]] == s, else -1); partner[s] == s leaves s
 * unmixed, i.e. row and column s of T_k hold a single 1 (PAPER.md:66 generalised: T_k stays
 * symmetric and doubly stochastic).  Odd S is fine.  ORACLE_NO_MIX is ignored here (pass the
 * identity instead).  Diagnostics as above; gap[s] == 0 exactly for an unmixed member.       */
int hadpsgd_oracle_step_matching(int S, int G, int64_t P,
                                 const void* grads, int grad_dtype,
                                 float* w, float* v,
                                 float lr, float mu, const int32_t* partner /*[S]*/, uint32_t flags,
                                 double* diag /* [3*S] or NULL */);
int hadpsgd_oracle_step_matching_f64(int S, int G, int64_t P,
                                     const void* grads, int grad_dtype,
                                     double* w, double* v,
                                     double lr, double mu, const int32_t* partner /*[S]*/, uint32_t flags);
/* Dense T for such a matching: T[s][s] = 1 if partner[s] == s, else T[s][s] = T[s][p] = 0.5. */
int hadpsgd_oracle_mixing_matrix_matching(int S, const int32_t* partner /*[S]*/, double* T /*[S*S]*/);

/* The same algorithm carried in double (state in double, gradients widened
 * exactly).  Used by the closed-form pins and to derive the fp32 tolerance.  */
int hadpsgd_oracle_step_f64(int S, int G, int64_t P,
                            const void* grads, int grad_dtype,
                            double* w, double* v,
                            double lr, double mu, uint64_t step_k, uint32_t flags);

/* bf16 working copy of fp32 weights for mixed-precision learners (
 * not in the paper): out[i] = the bf16 value NEAREST to w[i], ties to the value whose last
 * mantissa bit is even (IEEE round-to-nearest-even to 8 significant bits), written out as the
 * definition: the two bf16 neighbours of w[i] are compared by exact distance.  NaN -> a quiet
 * NaN, +-Inf unchanged, overflow past the largest finite bf16 -> +-Inf.  out holds bf16 bit
 * patterns (uint16).                                                                          */
int hadpsgd_oracle_round_bf16(int64_t n, const float* w, uint16_t* out);

/* Consensus distance D = sum_s sum_i (w[s][i] - mean_s w[.][i])^2 in double
 * (repeated mixing drives all learners to (1/n) sum theta^i).   */
int hadpsgd_oracle_consensus_distance(int S, int64_t P, const float* w, double* out);

#ifdef __cplusplus
}
#endif
#endif
