/*
 * nbody_b200.h -- C ABI of libnbody_b200.so: all-pairs softened gravity on one NVIDIA B200 (sm_100a).
 *
 * What is computed (arXiv astro-ph/0703100, Hamada & Iitaka, "The Chamomile Scheme"; citations are
 * to /root/reference/PAPER.md by line):
 *
 *     a_i   =  sum_j m_j r_ij / (r_ij^2 + eps^2)^(3/2),   r_ij = r_j - r_i      Eq. (1)
 *     phi_i = -sum_j m_j / (r_ij^2 + eps^2)^(1/2)                               Fig. A.4
 *
 * with G = 1, in FP32 arithmetic with an approximate reciprocal square root, as in the paper's
 * pipeline description (Fig. A.3: all variables are float, r1i = 1/sqrt(r2)).
 * A pair whose three coordinate differences are all exactly zero (in particular i == j when the
 * i-set is the j-set) contributes nothing to a_i and nothing to phi_i (reading R1).
 * The sum over j is formed as the paper's Eq. (2): partial sums over blocks of
 * consecutive j-particles, each started from zero, added to a running total.
 *
 * The call shape follows the paper's only entry point, force(xj, mj, xi, eps2, a, ni, nj)
 * (PAPER.md:235, 246, 376-382): separate i- and j-sets, so that the same call serves direct
 * integration (i-set == j-set) and active subsets / tree interaction lists.
 *
 * Conventions for every function below
 *   - plain C, no C++ types; safe to call through ctypes / dlopen.
 *   - "device" pointers are CUDA global-memory pointers valid on the current device; "host"
 *     pointers are ordinary process memory.  The library never takes ownership of any argument.
 *   - counts are int64_t and must be in [0, 2^31 - 4097] (32-bit particle indices inside the kernels).
 *   - every function returns an nb_status (int); nothing throws, aborts or prints.
 *   - functions that take a stream enqueue work on it and return without synchronising; results
 *     are valid once the stream has reached that point.  `stream` is a cudaStream_t passed as
 *     void*; NULL means the legacy default stream.
 *   - results are bitwise reproducible for the same inputs, device and library build (no floating
 *     point atomics; all reductions run in a fixed order).
 *   - there is no CPU fallback and no other GPU architecture: a device whose compute capability
 *     is not 10.x yields NB_ERR_UNSUPPORTED_DEVICE.
 *   - threads: the library may be called from several host threads.  Error and launch-count state is per thread.  The
 *     internal workspace is per (device, stream) and is locked while a call grows it and enqueues the work that uses
 *     it, so calls that share a stream (all *_host calls share the default stream) are serialised on the host; their
 *     device work runs in stream order, as always.  nb_release_workspace / nb_release_stream must not run while
 *     another thread is inside a call on that device / stream.
 *   - CUDA graphs: once the workspace of a stream is warm (one call of the same or a larger shape has run on it) a call
 *     enqueues kernels only and can be captured.  A captured graph holds the workspace's addresses: replaying it after
 *     a LARGER call on the same stream (which re-allocates the buffers it grows), after nb_release_workspace or after
 *     nb_release_stream reads freed memory -- capture again after any of these.
 *   - coordinate range of the coincident-pair rule: the kernels run flush-to-zero, so a pair whose three coordinate
 *     differences are all SUBNORMAL (|d| < 2^-126) may count as coincident, and whether it does can depend on the
 *     decomposition.  With every coordinate either 0 or >= 2^-102 in magnitude all non-zero differences are normal
 *     numbers and the rule is exactly "all three differences are zero" (tests/test_force_gpu.py bounds this).
 *   - the library reads no environment variable on any call; its debugging switches are in nb_debug.h.
 */
#ifndef NBODY_B200_H
#define NBODY_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum nb_status {
    NB_OK = 0,
    NB_ERR_INVALID_VALUE = 1,      /* negative / too large count, required pointer NULL, eps2 < 0 or not finite, ... */
    NB_ERR_CUDA = 2,               /* a CUDA runtime call failed; see nb_last_cuda_error() */
    NB_ERR_ALLOC = 3,              /* the internal workspace could not be allocated */
    NB_ERR_UNSUPPORTED_DEVICE = 4, /* current device is not compute capability 10.x */
    NB_ERR_LIMIT = 5               /* the call exceeds the fixed limit of a no-allocation entry point (nb_force_noalloc) */
} nb_status;

/*
 * nb_force -- Eq. (1) and phi for n_i i-particles against n_j j-particles.
 *
 *   n_i      number of i-particles (particles that receive a force)
 *   x_i      device, const, float [n_i][3]   positions (x,y,z) of the i-particles, 4-byte aligned
 *   n_j      number of j-particles (particles that exert a force)
 *   x_j      device, const, float [n_j][3]   positions of the j-particles
 *   m_j      device, const, float [n_j]      masses of the j-particles
 *   eps2     softening length SQUARED ("eps2"), >= 0 and finite
 *   acc_out  device, float [n_i][3]          receives a_i; required when n_i > 0
 *   pot_out  device, float [n_i]             receives phi_i; may be NULL (phi is then not stored)
 *   stream   cudaStream_t as void*
 *
 * x_i may alias x_j (i-set == j-set).  acc_out / pot_out must not overlap any input.
 * n_i == 0: NB_OK, nothing is written.  n_j == 0: NB_OK, outputs are zero-filled.
 * Inputs are not validated on the device: non-finite or |x| > ~1e18 inputs give undefined values.
 * Uses an internal per-stream workspace (packed j records, j-split partial sums) that grows on
 * demand with stream-ordered allocation; once warm the call is CUDA-graph capturable (see "CUDA graphs" above).
 * Calls with few i-particles (n_i <= 512 up to 2^26 pairs, n_i <= 4096 up to 2^25 pairs, n_i <= 32 up to 2^29 pairs: BASELINE.json configs[0] and
 * [2]) run as ONE launch of the small-i-set kernel (packed over j; the j-split is summed through lanes, warps, a
 * thread-block cluster or ticketed FP64 partials); larger ones as pack (+ coincidence pre-pass) + force kernel (+ second pass).
 */
int nb_force(int64_t n_i, const float *x_i,
             int64_t n_j, const float *x_j, const float *m_j,
             float eps2,
             float *acc_out, float *pot_out,
             void *stream);

/*
 * nb_force_host -- the same operation on HOST arrays: copies the inputs to the device, runs
 * nb_force, copies a and phi back and waits for completion.  This is the paper's force() with its
 * steps (a) and (l) -- host->device and device->host transfers -- inside the call
 * (PAPER.md:151, 167, 233-237).  All pointers are host pointers with the layouts of nb_force.
 * Blocking.  pot_out may be NULL.
 */
int nb_force_host(int64_t n_i, const float *x_i,
                  int64_t n_j, const float *x_j, const float *m_j,
                  float eps2,
                  float *acc_out, float *pot_out);

/*
 * nb_leapfrog_kdk -- n_steps kick-drift-kick leapfrog steps with all state on the device.
 * (Not in the paper; BASELINE.json north_star bullet 4 and configs[4]; reading R8.)
 *
 *     a = force(x)                      once, before the first step
 *     repeat n_steps times:
 *         v += a * (dt/2);  x += v * dt;  a = force(x);  v += a * (dt/2)
 *
 *   n        number of particles (i-set == j-set == all)
 *   x, v     device, float [n][3], updated in place
 *   m        device, const, float [n]
 *   eps2     softening squared, >= 0, finite;   dt  finite;   n_steps >= 0
 *   acc_io   device, float [n][3]: receives a at the final time (its content on entry is ignored)
 *   pot_out  device, float [n]: receives phi at the final time; may be NULL
 *
 * n_steps == 0 only evaluates a and phi of the given state.
 * Small systems (n <= 32768) with n_steps >= 64: the identical middle steps are captured into a CUDA graph (eight steps per
 * graph) and replayed -- the same launches, the same bits (nb_debug.h: NB_STEP_GRAPH=0 switches it off).  A default stream
 * (NULL / legacy or per-thread) cannot be captured: the run is then enqueued on a private non-blocking stream of the device
 * that first waits for the work already enqueued on the caller's stream, and the caller's stream waits for the run before
 * anything enqueued after the call -- the stream order the caller sees is unchanged.  nb_hermite4 does the same.
 */
int nb_leapfrog_kdk(int64_t n, float *x, float *v, const float *m,
                    float eps2, float dt, int64_t n_steps,
                    float *acc_io, float *pot_out,
                    void *stream);

/*
 * nb_kick_drift / nb_kick -- the O(n) updates of the KDK leapfrog on their own (the kernels nb_leapfrog_kdk runs between its
 * force evaluations), for drivers that own only a SLICE of the particles: the i-sharded multi-GPU integration of
 * DESIGN.md section 8 calls them on each rank's slice around the all-gather + nb_force_packed of every step.
 *
 *     nb_kick_drift:  v += acc * h  (n_kicks = 1)  or  v += acc * h; v += acc * h  (n_kicks = 2: the closing half-kick of one
 *                     step and the opening half-kick of the next, two separately rounded FMAs);  then  x += v * dt
 *     nb_kick:        v += acc * h
 *
 *   x, v  device, float [n][3], updated in place      acc  device, const, float [n][3]      h, dt finite
 */
int nb_kick_drift(int64_t n, float *x, float *v, const float *acc, float h, int n_kicks, float dt, void *stream);
int nb_kick(int64_t n, float *v, const float *acc, float h, void *stream);

/*
 * nb_force_jerk -- force + jerk + potential for the 4th-order Hermite scheme: the paper's second
 * pipeline description (Fig. A.2, Fig. A.4; used by the authors'
 * Hermite code):
 *
 *     a_i    =  sum_j m_j d / r^3                          d = r_j - r_i,  r^2 = d.d + eps2
 *     jerk_i =  sum_j m_j [ dv / r^3 - 3 (d.dv) d / r^5 ]  dv = v_j - v_i      (= d a_i / dt)
 *     phi_i  = -sum_j m_j / r
 *
 *   x_i, v_i  device, const, float [n_i][3]   positions and velocities of the i-particles
 *   x_j, v_j  device, const, float [n_j][3]   positions and velocities of the j-particles
 *   m_j       device, const, float [n_j]
 *   acc_out, jerk_out   device, float [n_i][3], required when n_i > 0
 *   pot_out   device, float [n_i], may be NULL
 *
 * Everything else (aliasing, edge sizes, coincident-pair rule -- decided on the POSITIONS only --,
 * asynchrony, errors, reproducibility) is as for nb_force.
 */
int nb_force_jerk(int64_t n_i, const float *x_i, const float *v_i,
                  int64_t n_j, const float *x_j, const float *v_j, const float *m_j,
                  float eps2,
                  float *acc_out, float *jerk_out, float *pot_out,
                  void *stream);

/*
 * nb_force_packed -- nb_force for a caller that already holds the j-particles as packed 16-byte records
 * (x, y, z, m): the paper's own internal layout, p_xj[j][0..3] = (x, y, z, m) (Fig. A.1), so the
 * packing pass (row a1) is skipped.  This is the entry the multi-GPU i-sharding uses: every rank all-gathers the
 * packed records of all ranks' particles and evaluates its own i-slice against them.
 *
 *   xm_j   device, const, float [n_j][4] = (x, y, z, m) per j-particle, 16-byte aligned
 * Everything else as for nb_force.  A record with m = 0 adds nothing (padding of a ragged shard).
 */
/* nb_pack_j -- row a1 on its own: (x, y, z) || m -> xm_out [n_j][4], device, 16-byte aligned (Fig. A.1). */
int nb_pack_j(int64_t n_j, const float *x_j, const float *m_j, float *xm_out, void *stream);

int nb_force_packed(int64_t n_i, const float *x_i,
                    int64_t n_j, const float *xm_j,
                    float eps2,
                    float *acc_out, float *pot_out,
                    void *stream);

/*
 * nb_force_eps_i -- nb_force with the softening carried PER i-PARTICLE, as in the paper's own driver, where slot 3
 * of every i-record is eps2 (Fig. A.1: p_xi[i][3] = eps2; Fig. A.3 PAPER.md:446-450:
 * eps2 = INPUT_I[3]) -- the first step of the generalised CUNBODY-1 kernel of section 4.5:
 *
 *     a_i = sum_j m_j d / (d.d + eps2_i[i])^(3/2),   phi_i = -sum_j m_j / (d.d + eps2_i[i])^(1/2)
 *
 *   eps2_i   device, const, float [n_i], every value >= 0 and finite (not validated: device data)
 * Everything else as for nb_force.  Coincident pairs add nothing whatever eps2_i is (0 included).
 */
int nb_force_eps_i(int64_t n_i, const float *x_i, const float *eps2_i,
                   int64_t n_j, const float *x_j, const float *m_j,
                   float *acc_out, float *pot_out,
                   void *stream);

/*
 * nb_cunbody_force / nb_cunbody_force_jerk_pot -- the paper's own library call, cunbody_api(p_xj, p_xi, p_fi, ni, nj)
 * (PAPER.md:389, 420), for its two pipeline descriptions, run by the generalised pair kernel of section 4.5
 * (include/nb_pipeline.cuh, where users instantiate their own pipelines the same way):
 *
 *   nb_cunbody_force           Fig. A.1 / A.3
 *        p_xj [nj][4] = (x, y, z, m)       p_xi [ni][4] = (x, y, z, eps2)       p_fi [ni][3] = (ax, ay, az)
 *   nb_cunbody_force_jerk_pot  Fig. A.2 / A.4; eps2 is the listing's constant 1/256^2
 *        p_xj [nj][7] = (x, v, m)          p_xi [ni][6] = (x, v)                p_fi [ni][7] = (a, jerk, pot)
 *
 * All rows are DEVICE float arrays (the paper passes host doubles and copies inside; here the caller owns device
 * memory, as for nb_force).  p_fi is overwritten, not accumulated into.  Coincident pairs add nothing (reading R1).
 * These entry points run the listings as written (scalar FP32, any pipeline); nb_force / nb_force_eps_i /
 * nb_force_jerk compute the same sums with the specialised kernels and are 1.8x faster (N = 131072).
 */
int nb_cunbody_force(const float *p_xj, const float *p_xi, float *p_fi, int64_t ni, int64_t nj, void *stream);
int nb_cunbody_force_jerk_pot(const float *p_xj, const float *p_xi, float *p_fi, int64_t ni, int64_t nj, void *stream);

/*
 * nb_cunbody_lennard_jones -- the same cunbody_api call for a central force other than gravity: the paper lists
 * "van der Waals molecular interactions" among the interactions of its generalised library (section 4.5,
 * PAPER.md:363) without a formula; reading R19 takes the 12-6 Lennard-Jones pair with Lorentz-Berthelot
 * mixing, all pairs, no cut-off, with d = r_j - r_i, r2 = d.d, sigma = sigma_i/2 + sigma_j/2,
 * eps = sqrt(eps_i) sqrt(eps_j), s6 = (sigma^2 / r2)^3:
 *
 *     F_i = - sum_j 24 eps (2 s6^2 - s6) / r2 * d          U_i = sum_j 4 eps (s6^2 - s6)
 *
 *        p_xj [nj][5] = (x, y, z, sigma_j / 2, sqrt(eps_j))       p_xi [ni][5] likewise       p_fi [ni][4] = (Fx, Fy, Fz, U)
 *
 * F_i is the force ON particle i; the total energy of a closed system is 1/2 sum_i U_i.  DEVICE float rows, p_fi
 * overwritten, coincident pairs add nothing, errors as for nb_cunbody_force.
 */
int nb_cunbody_lennard_jones(const float *p_xj, const float *p_xi, float *p_fi, int64_t ni, int64_t nj, void *stream);

/*
 * nb_force_batched -- many independent small (i-set, j-set) sub-problems of nb_force in ONE launch:
 * the use the paper shapes its interface for, a host tree code calling the force routine on
 * interaction lists of "several thousands" particles per group (PAPER.md:246 last sentence, section
 * 4.4 PAPER.md:355-359).  Sub-problem b = i-particles [i_offsets[b], i_offsets[b+1]) of x_i against
 * j-particles [j_offsets[b], j_offsets[b+1]) of x_j / m_j (CSR-style concatenation):
 *
 *     for b in 0 .. n_batch-1:   nb_force(n_i(b), x_i + 3 i_offsets[b], n_j(b), x_j + 3 j_offsets[b],
 *                                         m_j + j_offsets[b], eps2, acc_out + 3 i_offsets[b], pot_out + i_offsets[b])
 *
 *   n_batch    number of sub-problems
 *   i_offsets  device, const, int32 [n_batch + 1], non-decreasing, i_offsets[n_batch] <= n_i_total
 *   j_offsets  device, const, int32 [n_batch + 1], non-decreasing, j_offsets[n_batch] <= n_j_total
 *   n_i_total, n_j_total   lengths of the concatenated arrays (host values; the offsets are NOT read on the host)
 *   x_i [n_i_total][3], x_j [n_j_total][3], m_j [n_j_total], acc_out [n_i_total][3], pot_out [n_i_total] or NULL: device
 *
 * Each sub-problem is handled by ceil(n_i(b) / tile) CTAs (tile = 64 .. 512, chosen from the mean
 * n_i_total / n_batch) whose 8 warps split its j-range; no partial sums leave a CTA.  A sub-problem with
 * n_j(b) == 0 gets zeros; i-particles outside every sub-problem are not written.  The offsets are not
 * validated.  Same coincident-pair rule, determinism and error conventions as nb_force.
 */
int nb_force_batched(int64_t n_batch, const int32_t *i_offsets, const int32_t *j_offsets,
                     int64_t n_i_total, const float *x_i,
                     int64_t n_j_total, const float *x_j, const float *m_j,
                     float eps2,
                     float *acc_out, float *pot_out,
                     void *stream);

/*
 * nb_force_batched_packed -- nb_force_batched for a caller that keeps the interaction-list records on the device as packed
 * 16-byte (x, y, z, m) rows (the batched analogue of nb_force_packed; the paper's own layout, Fig. A.1):
 * no pack pass -- on tree lists that pass moves 32 B per list entry per call, 5-6 % of a call -- and a host caller ships
 * 16 B per entry once instead of re-sending (x, y, z) and m.  xm_j: device, const, float [n_j_total][4], 16-byte aligned.
 * Same results as nb_force_batched on the same records, bit for bit; everything else as there.
 */
int nb_force_batched_packed(int64_t n_batch, const int32_t *i_offsets, const int32_t *j_offsets,
                            int64_t n_i_total, const float *x_i,
                            int64_t n_j_total, const float *xm_j,
                            float eps2,
                            float *acc_out, float *pot_out,
                            void *stream);

/*
 * nb_force_batched_indexed -- nb_force_batched with the interaction lists given as INDICES into one array of packed particle
 * records: what a tree code holds (its particles and cell pseudo-particles once, a list of integers per group).  Sub-problem
 * b: i-particles as in nb_force_batched; j-list = xm_p[j_index[k]] for k in [j_offsets[b], j_offsets[b+1]).  4 bytes per list
 * entry instead of 16 cross PCIe / HBM; the kernel fills its shared-memory rings with gathered 16-byte asynchronous copies.
 *
 *   j_index   device, const, int32 [n_list_total], every value in [0, n_p) (not validated: device data)
 *   xm_p      device, const, float [n_p][4] = (x, y, z, m), 16-byte aligned
 * Same results as nb_force_batched on the expanded lists, bit for bit; everything else as there.
 */
int nb_force_batched_indexed(int64_t n_batch, const int32_t *i_offsets, const int32_t *j_offsets,
                             int64_t n_i_total, const float *x_i,
                             int64_t n_list_total, const int32_t *j_index,
                             int64_t n_p, const float *xm_p,
                             float eps2,
                             float *acc_out, float *pot_out,
                             void *stream);

/*
 * nb_hermite4 -- n_steps steps of the 4th-order Hermite scheme with a shared, constant time step, all state on the
 * device: the scheme the paper names as the user of its force + jerk pipeline; the paper does
 * not describe it, this is the textbook predict - evaluate - correct form with one nb_force_jerk per step:
 *
 *     a, j = force_jerk(x, v)                                          once, before the first step
 *     repeat n_steps times:
 *         xp = x + v dt + a dt^2/2 + j dt^3/6;   vp = v + a dt + j dt^2/2
 *         a1, j1 = force_jerk(xp, vp)
 *         v' = v + (a + a1) dt/2 + (j - j1) dt^2/12;   x' = x + (v + v') dt/2 + (a - a1) dt^2/12
 *         x, v, a, j <- x', v', a1, j1
 *
 *   x, v      device, float [n][3], updated in place          m   device, const, float [n]
 *   acc_io, jerk_io   device, float [n][3]: receive the a and j carried out of the last step (evaluated at its
 *             predicted state); their content on entry is ignored
 *   pot_out   device, float [n] or NULL: phi of the last evaluation
 * n_steps == 0 only evaluates a, j and phi of the given state.
 */
int nb_hermite4(int64_t n, float *x, float *v, const float *m,
                float eps2, float dt, int64_t n_steps,
                float *acc_io, float *jerk_io, float *pot_out,
                void *stream);

/*
 * nb_hermite4_block_step -- ONE block step of the 4th-order Hermite scheme with individual (block) time steps: the
 * active-subset integration that BASELINE.json configs[2] is shaped for (i-set = the particles due now, j-set =
 * everybody), on top of the separate i- and j-sets of the paper's call.  The paper names the Hermite
 * scheme as the user of its force + jerk pipeline and does not describe it; this is the textbook
 * form (reading R20).  Every particle k holds (x, v, a, j) at its OWN time t[k] <= t_now:
 *
 *     all k:          h = t_now - t[k];  xp = x + v h + a h^2/2 + j h^3/6;  vp = v + a h + j h^2/2
 *     active i only:  a1, j1 = force_jerk(i-set = (xp, vp) of the active, j-set = (xp, vp, m) of all n)
 *                     v' = v + (a + a1) h/2 + (j - j1) h^2/12;   x' = x + (v + v') h/2 + (a - a1) h^2/12
 *                     x, v, a, j, t <- x', v', a1, j1, t_now
 *
 *   x, v, acc_io, jerk_io   device, float [n][3]: state at t[k]; the active rows are updated in place, no other row
 *             is written          m   device, const, float [n]
 *   t         device, double [n]: each particle's own time; the active entries become t_now.  h is formed in double
 *             and rounded to float once (exact for the usual power-of-two step hierarchy)
 *   active    device, const, int32 [n_act]: DISTINCT indices in [0, n), any order; not validated on the device
 *             (out-of-range or repeated indices: undefined results).  n_act == 0: success, nothing is touched
 *   t_now     the block time.  Who is due and each particle's next step are the caller's business.
 * Asynchronous on `stream`; 2 small launches + those of one nb_force_jerk(n_act, n) without phi.
 */
int nb_hermite4_block_step(int64_t n, float *x, float *v, const float *m,
                           float *acc_io, float *jerk_io, double *t,
                           int64_t n_act, const int32_t *active, double t_now,
                           float eps2, void *stream);

/*
 * nb_block_schedule -- the scheduler's question for nb_hermite4_block_step: when is the next block step and who is due
 * (reading R20; the paper has no integrator).  With due_k = t[k] + dt[k] (one FP64 addition):
 *
 *     t_next = min_k due_k          active = { k : due_k == t_next } in ASCENDING index order
 *
 *   t, dt       device, const, double [n]: each particle's own time and its current step
 *   t_next_out  device, double [1]         active_out  device, int32 [n] (only the first n_act entries are written)
 *   n_act_out   device, int32 [1]: the caller reads it back (4 bytes) to size the nb_hermite4_block_step call
 * Index work: exact and deterministic (no floating-point atomics, ordered compaction).  n == 0: t_next = +inf, n_act = 0.
 * A due time that is not finite (t + dt = +-inf or NaN: e.g. a particle parked with dt = +inf) takes no part: it is never the
 * minimum and never due; if no due time is finite, t_next = +inf and n_act = 0.  Asynchronous on `stream`.
 */
int nb_block_schedule(int64_t n, const double *t, const double *dt,
                      double *t_next_out, int32_t *active_out, int32_t *n_act_out,
                      void *stream);

/*
 * nb_block_step_size -- the Aarseth step-size criterion of the block Hermite scheme (textbook; reading R20),
 * per particle, from its two evaluations (a0, j0) at t and (a1, j1) at t + h:
 *
 *     a2 = (-6 (a0 - a1) - h (4 j0 + 2 j1)) / h^2       a3 = (12 (a0 - a1) + 6 h (j0 + j1)) / h^3
 *     a2' = a2 + h a3          dt = sqrt( eta (|a1| |a2'| + |j1|^2) / (|j1| |a3| + |a2'|^2) )
 *
 * The value feeds an integer decision (the block level = its power-of-two quantisation, the caller's), so the arithmetic
 * is pinned: FP32, every operation one IEEE round-to-nearest operation in the order written (da = a0 - a1;
 * s1 = 4 j0 + 2 j1; a2 = -(6 da + h s1) / (h h); s2 = j0 + j1; a3 = (12 da + (6 h) s2) / ((h h) h); a2' = a2 + h a3;
 * |z|^2 = (x x + y y) + z z; top = sqrt|a1|^2 sqrt|a2'|^2 + |j1|^2; bot = sqrt|j1|^2 sqrt|a3|^2 + |a2'|^2;
 * dt = sqrt(eta (top / bot))): bit-identical to the oracle's numpy float32 definition.
 *
 *   a0, j0, a1, j1   device, const, float [n][3]      h   device, const, float [n] (> 0)
 *   eta   > 0, finite                                 dt_out   device, float [n]
 * bot == 0 (a particle with constant acceleration) gives +inf or NaN as IEEE arithmetic says.  Asynchronous on `stream`.
 */
int nb_block_step_size(int64_t n, const float *a0, const float *j0, const float *a1, const float *j1,
                       const float *h, float eta, float *dt_out, void *stream);

/*
 * nb_force_jerk_host -- nb_force_jerk on HOST arrays: the paper's force() of Fig. A.2 with its
 * host->device and device->host copies (steps (a) and (l)) inside the call.  Blocking.
 */
int nb_force_jerk_host(int64_t n_i, const float *x_i, const float *v_i,
                       int64_t n_j, const float *x_j, const float *v_j, const float *m_j,
                       float eps2,
                       float *acc_out, float *jerk_out, float *pot_out);

/* nb_plan_query for nb_force_jerk (same out[] layout; K <= 4, 256 j-particles of 32 bytes per stage). */
int nb_plan_query_jerk(int64_t n_i, int64_t n_j, int sm_count, int64_t out[8]);

/*
 * nb_plan_query -- the decomposition the launch planner picks for (n_i, n_j) on a device with
 * sm_count SMs (pure host function, no CUDA call; sm_count <= 0 means 148).
 * out[0] = K  i-particles per thread        out[1] = WI warps per CTA along i
 * out[2] = WJ warps per CTA along j         out[3] = S  j-chunks across CTAs (grid.y)
 * out[4] = number of i-tiles (grid.x)       out[5] = i-particles per CTA tile (32*K*WI)
 * out[6] = j-particles per shared-memory stage  out[7] = pipeline stages
 */
int nb_plan_query(int64_t n_i, int64_t n_j, int sm_count, int64_t out[8]);

/* Number of kernel launches the most recent nb_force / nb_leapfrog_kdk / nb_force_host call of this thread enqueued. */
int64_t nb_last_launch_count(void);

/*
 * nb_profile_enable / nb_profile_read -- optional timing of the dominant kernel (the pair-interaction
 * kernel, rows a2..a7) for the roofline report.  While enabled, every force-kernel launch of this
 * thread is bracketed by two CUDA events recorded on the launching stream.  nb_profile_read waits
 * for the recorded events, returns the number of bracketed launches and the sum of their durations in
 * milliseconds, and clears the record.  Disabled by default; when disabled nothing is recorded.
 */
int nb_profile_enable(int on);
int nb_profile_read(int64_t *n_launches, double *total_ms);

/* nb_plan_query for the small-i-set kernel nb_force uses for few i-particles (csrc/nb_small.cuh):
 * out[0] = NW warps per CTA (8 or 16)       out[1] = KI i-particles per thread
 * out[2] = LJ lanes of a warp along j (32 / LJ along i)      out[3] = WJ warps per CTA along j
 * out[4] = S  j-chunks across CTAs (grid.y) out[5] = CS CTAs per thread-block cluster
 * out[6] = number of i-tiles (grid.x); i-particles per CTA tile = (NW / WJ) * KI * (32 / LJ)
 * out[7] = 1 if nb_force takes this kernel for (n_i, n_j) by default */
int nb_plan_query_small(int64_t n_i, int64_t n_j, int sm_count, int64_t out[8]);
/* The same for the small-i-set force + jerk kernel (csrc/nb_small_hermite.cuh; KI = 1): out[7] bit 0 = nb_force_jerk takes
 * it for (n_i, n_j) by default (up to 2^25 pairs, more for narrow i-sets; the kernel packs the j-records itself), bit 1 = nb_hermite4 and
 * nb_hermite4_block_step do (up to 2^22 pairs, 2^23 for at most 512 active particles; their predictor has packed the records). */
int nb_plan_query_small_jerk(int64_t n_i, int64_t n_j, int sm_count, int64_t out[8]);

/* Frees every internal workspace of the current device (synchronises the device). */
int nb_release_workspace(void);

/* Frees the workspace kept for `stream` on the current device (waits for that stream first).  Call it before destroying a
 * stream the library has been used on: the workspace is keyed by the stream handle and would otherwise stay allocated
 * until nb_release_workspace -- and be inherited by a later stream that happens to get the same handle. */
int nb_release_stream(void *stream);

/*
 * nb_force_noalloc -- nb_force for callers that must not allocate device memory (a serving loop, a harness that forbids
 * cudaMalloc, code under stream capture): the same operation, arguments, layouts, results and error behaviour as nb_force
 * (Eq. (1) and phi; the one-launch small-i-set kernel, j-split of section 4.2), with
 *
 *   - n_i <= NB_NOALLOC_MAX_I, else NB_ERR_LIMIT and nothing is launched or written (any n_j nb_force accepts);
 *   - NO device allocation, ever: the call makes no cudaMalloc / cudaMallocAsync / cudaFree and uses no library routine
 *     that allocates.  The scratch of the j-split (FP64 partial sums [n_i][groups] + one ticket counter per i-tile slice)
 *     lives in ONE static __device__ array of NB_NOALLOC_SCRATCH_BYTES inside the library: every GPU that loads the
 *     library holds it from load until the process exits, whether or not this entry point is ever called.  When the
 *     planner's j-split would need more partial sums than the array holds, the call runs with fewer j-chunks (slower,
 *     same result up to summation order).
 *
 * Sharing: ALL calls on a device -- from any thread, on any stream -- use the same array, which keeps the last call's
 * contents.  Every call clears the ticket counters it will use first (stream-ordered, on `stream`); the partial sums are
 * written before they are read.  Two nb_force_noalloc calls that OVERLAP on the GPU (different streams, or two host
 * threads on different streams) race on the array and give undefined results: serialise them (one stream, or events).
 * Calls on one stream never overlap.  nb_force and every other entry point use their own workspace and are not affected.
 *
 * The first call on each device does the one-time set-up (resolves the array's device address, raises the kernel's
 * shared-memory limit): make it outside any stream capture.  The debugging switches of nb_debug.h do not apply.
 * Results: bit for bit nb_force's when nb_force takes the small-i-set kernel for the shape and the j-split is not
 * reduced; within the library's tolerance (BASELINE.json north_star: acc RMS 1e-5, max 1e-4, phi RMS 1e-5) otherwise.
 */
#define NB_NOALLOC_MAX_I 4096
#define NB_NOALLOC_SCRATCH_BYTES (131072 * 32 + 4096 * 4)   /* 4 MiB of partial sums + 16 KiB of ticket counters */
int nb_force_noalloc(int64_t n_i, const float *x_i,
                     int64_t n_j, const float *x_j, const float *m_j,
                     float eps2, float *acc_out, float *pot_out, void *stream);

const char *nb_status_string(int status);   /* static storage */
int nb_last_cuda_error(void);                /* cudaError_t behind this thread's last NB_ERR_CUDA / NB_ERR_ALLOC */
int nb_version(void);                        /* major*10000 + minor*100 + patch */

#ifdef __cplusplus
}
#endif
#endif /* NBODY_B200_H */
