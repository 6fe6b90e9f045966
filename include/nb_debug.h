/*
 * nb_debug.h -- debugging switches of libnbody_b200.so.  NOT part of the product contract of nbody_b200.h: nothing here
 * is needed to use the library, every switch only selects among code paths that compute the same thing (most of them
 * bit for bit), and the tests use them to reach each path on small inputs.
 *
 * The switches are process-wide.  They are read from the environment ONCE, when the library is first used (variables
 * of the same names), and can be changed afterwards only through nb_debug_set -- no library call reads the
 * environment on its hot path.  Setting a switch while another thread is inside a library call is a data race on
 * which path that call takes, nothing else.
 *
 *   key                value                      effect
 *   NB_PLAN            "K,WI,WJ,S"                decomposition of nb_force / nb_force_jerk (nb_plan_query's out[0..3])
 *   NB_SMALL           "0" | "1"                  never / always route nb_force through the small-i-set kernel
 *   NB_SMALL_PLAN      "NW,KI,LJ,WJ,S,CS"         decomposition of the small-i-set kernel (nb_plan_query_small's out[0..5])
 *   NB_SMALL_MASK      "exact" | "flag"           small-i-set kernel: mask every pair / only the pairs marked while staged
 *   NB_SMALL_JERK      "0" | "1"                  never / always route nb_force_jerk (and the Hermite steps) through the
 *                                                 small-i-set force + jerk kernel
 *   NB_SMALL_JERK_PLAN "NW,LJ,WJ,S,CS"            its decomposition (nb_plan_query_small_jerk's out[0], out[2..5])
 *   NB_SMALL_PDL       "0" | "1"                  small-i-set kernels (force, force + jerk): plain launch / programmatic stream serialisation (default)
 *   NB_MASK            "exact" | "bloom" | "list" where coincident pairs are found; also switches
 *                                                 the acceleration-only shortcut off
 *   NB_FUSED_REDUCE    "0" | "1"                  second pass of the j-split as a separate launch / inside the force kernel
 *   NB_DIRECT          "0"                        small calls go through nb_pack_j_kernel + TMA instead of packing in-kernel
 *   NB_STEP_GRAPH      "0"                        nb_leapfrog_kdk / nb_hermite4 enqueue every step eagerly (no CUDA graph)
 *   NB_HERMITE_FUSE    "0"                        nb_hermite4 corrects a step and predicts the next in two launches instead of one
 *   NB_BATCH_TILE      "64" | "128" | "256"       i-tile of nb_force_batched
 *
 * value == NULL or "" restores the default.  Returns NB_OK, or NB_ERR_INVALID_VALUE for an unknown key or a value that
 * does not parse (the switch is then left unchanged).
 */
#ifndef NB_DEBUG_H
#define NB_DEBUG_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

int nb_debug_set(const char *key, const char *value);

/* The decomposition make_plan is DEFINED by: the exhaustive search over every (K, WJ, S) (csrc/nb_plan.h).  Same out[]
 * layout as nb_plan_query; jerk != 0: the force + jerk family (K <= 4).  ~100 us: for tests of the fast planner only. */
int nb_debug_plan_exhaustive(int64_t n_i, int64_t n_j, int sm_count, int jerk, int64_t out[8]);

/* Number of plans computed (not served from the per-shape cache) by this process so far: nb_force-family calls only. */
int64_t nb_debug_plans_computed(void);

#ifdef __cplusplus
}
#endif
#endif /* NB_DEBUG_H */
