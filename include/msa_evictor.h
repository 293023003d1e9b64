/* msa_evictor.h -- C ABI of the computational-aware block evictor (host side, no GPU involved).
 *
 * SURVEY.md section 8 (f3).  The paper's Algorithm 1: every evictable KV-cache block B
 * carries the weight  f_B(t) * dT_B  (Eq. (3)) and the block with the smallest weight is
 * evicted, where
 *   dT_B   = 2*k5*pos_B + c0                 recomputation cost, Eq. (7); pos_B = number of
 *                                            tokens in front of the block in its sequence ("l1 + q1")
 *   f_B(t) = min( exp(-tau/alpha), exp(-(tau - tau0)/beta) ),  tau = t - (last access of B)      Eq. (9)
 * Each branch of f is a single exponential, so the ORDER of the branch weights of two blocks never changes
 * with t (order-preserving rule, Eq. (8)); the evictor keeps one ordered set per branch, keyed by the
 * time-independent part of the log weight, and all three operations are O(log n):
 *   log w1 = -t/alpha + [ last/alpha          + ln dT ]      log w2 = -t/beta + [ (last + tau0)/beta + ln dT ]
 * Evict takes the minimum of each set and returns argmin{ w1(B1), lambda * w2(B2) } (Algorithm 1, line 8).
 *
 * All functions are host-only and thread-compatible (one evictor per thread, or external locking).
 * Return value: MSA_OK (0) or a negative MSA_ERR_* code from msa.h.
 */
#ifndef MSA_EVICTOR_H_
#define MSA_EVICTOR_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct msa_evictor_s *msa_evictor;

typedef struct {
    double alpha;    /* decay time of the first branch of Eq. (9), > 0                              */
    double beta;     /* decay time of the second branch, 0 < beta (steeper: beta < alpha)           */
    double tau0;     /* horizontal shift of the second branch, >= 0                                 */
    double lambda;   /* Algorithm 1 line 8, > 0; 1 reproduces Eq. (9) exactly                       */
    double k5;       /* Eq. (7): dT = 2*k5*pos + c0 ...                                              */
    double c0;       /* ... with c0 = k2 - k3 + k5; dT must be > 0 for every block added            */
} msa_evictor_config;

/* Creates an empty evictor.  MSA_ERR_INVALID_ARG if a parameter is out of range or a pointer is NULL. */
int msa_evictor_create(const msa_evictor_config *cfg, msa_evictor *out);
void msa_evictor_destroy(msa_evictor ev);

/* Algorithm 1 "Add": block `block_id` became evictable (ref-count 0).  `position` = tokens in front of it in
 * its sequence, `last_access` = time of its last use (any monotone clock, same unit as alpha / beta / tau0).
 * MSA_ERR_INVALID_ARG: NULL, negative position, dT <= 0, non-finite time; MSA_ERR_OVERLAP: id already present. */
int msa_evictor_add(msa_evictor ev, int64_t block_id, int64_t position, double last_access);

/* Algorithm 1 "Remove": the block was hit (or is being evicted).  MSA_ERR_OUT_OF_RANGE if it is not present. */
int msa_evictor_remove(msa_evictor ev, int64_t block_id);

/* Algorithm 1 "Evict" at time t_now: removes and returns the block with the smallest weight, O(log n).
 * MSA_ERR_OUT_OF_RANGE if the evictor is empty. */
int msa_evictor_evict(msa_evictor ev, double t_now, int64_t *block_id);

/* The same decision by a linear scan over all blocks (the O(n) strategy the paper compares against,
 * PAPER.md:235); kept for the measurement and as a cross-check.  Removes the block it returns. */
int msa_evictor_evict_linear(msa_evictor ev, double t_now, int64_t *block_id);

/* Online adjustment of lambda: lambda = exp((tau - tau0)/beta - tau/alpha), Eq. (10), moves the
 * effective turning point of Eq. (9) to the observed lifespan tau; takes effect at the next evict, O(1). */
int msa_evictor_set_lambda(msa_evictor ev, double lambda);

/* Number of evictable blocks held. */
int64_t msa_evictor_size(msa_evictor ev);

/* min( w1, lambda*w2 ) of a block at time t_now (Eq. (3) with Eq. (9) when lambda = 1); NaN if absent. */
double msa_evictor_weight(msa_evictor ev, int64_t block_id, double t_now);

#ifdef __cplusplus
}
#endif
#endif /* MSA_EVICTOR_H_ */
