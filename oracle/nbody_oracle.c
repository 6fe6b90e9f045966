/*
 * nbody_oracle.c -- the CPU ORACLE for the all-pairs softened gravity path.
 *
 * TEST INFRASTRUCTURE, NOT PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call anything in oracle/.  The CUDA
 * path (paper_astro_ph_0703100_b200/csrc) shares no code, header, table or helper with this file
 * and neither side includes or imports the other.
 *
 * What it is: the *definition* of the result, written out in double precision, plain loops, no
 * blocking, no fusion, no reordering.  The method of the paper (the Chamomile Scheme) reaches
 * exactly this sum, up to FP32 rounding order, just faster; so the oracle is Eq. (1) itself:
 *
 *     a_i = sum_j  m_j r_ij / (r_ij^2 + eps^2)^(3/2),     r_ij = r_j - r_i      PAPER.md:30-32, Eq. (1)
 *     phi_i = - sum_j m_j / (r_ij^2 + eps^2)^(1/2)                              PAPER.md:509-516, 552 (Fig. A.4:
 *                                                     mf = mj*r5i*r2, pot = mf*r2 = mj/sqrt(r2), OUTPUT[6] -= pot)
 *
 * with G = 1 (absent from Eq. (1)), the softening passed as eps^2 (PAPER.md:227, 235, 379:
 * "eps2"), and per-pair steps in the order of the paper's pipeline description
 * (Fig. A.3): d = r_j - r_i; r2 = d.d + eps2; r1i = 1/sqrt(r2); r2i, r3i;
 * mr3i = m_j r3i; a += mr3i d.
 *
 * Reading taken where the paper is silent (reading R1): a pair whose three coordinate
 * differences are all exactly zero ("coincident", which includes i == j when the i-set is the
 * j-set) contributes nothing to a_i and nothing to phi_i.  Eq. (1) has no i != j test and the
 * unmasked pipeline would add -m_i/eps to phi_i (and 0*inf = NaN when eps = 0).
 *
 * Accumulation: one double accumulator per component, j ascending.  With n_j <= 2^20 the rounding
 * error of that sum is <~ n_j 2^-53 ~ 1e-10 of the summand scale, five orders below the FP32
 * tolerances the CUDA path is held to, so no compensated summation is used.
 *
 * The leapfrog is the textbook kick-drift-kick scheme (not in the paper; BASELINE.json
 * north_star bullet 4, configs[4]; reading R8):
 *     a0 = force(x0);  per step:  v += a dt/2;  x += v dt;  a = force(x);  v += a dt/2.
 *
 * Pins (tests/test_oracle_pins.py): exact two-body rationals, coincident rule, momentum
 * antisymmetry, translation / rotation / axis-permutation invariance, Plummer and uniform-sphere
 * potential energies, brute force in exact rational arithmetic at N <= 8, large-eps limit, regular
 * figures, softened circular binary, time reversal, dt^2 convergence, a = -grad(phi), Newton's shell theorems,
 * superposition.
 * Parity unpinned: nothing in this file.  (The *value* of C4's energy drift is not pinned by the
 * paper -- see DESIGN.md -- but that is a property of the FP32 path, not an oracle function.)
 *
 * Build: gcc -O2 -fopenmp -ffp-contract=off -fPIC -shared (oracle/__init__.py: build()).  No -ffast-math.
 * OpenMP only parallelises the independent i-loop; the j-loop is sequential and ordered.
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void oracle_set_num_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* One i-particle against all j, Eq. (1) and phi, double precision.  out4 = (ax, ay, az, phi). */
static void one_i(const double xi[3], int64_t n_j, const double *xj, const double *mj, double eps2,
                  double out4[4])
{
    double ax = 0.0, ay = 0.0, az = 0.0, phi = 0.0;
    for (int64_t j = 0; j < n_j; ++j) {
        double dx = xj[3 * j + 0] - xi[0];            /* r_ij = r_j - r_i  */
        double dy = xj[3 * j + 1] - xi[1];
        double dz = xj[3 * j + 2] - xi[2];
        if (dx == 0.0 && dy == 0.0 && dz == 0.0)      /* coincident pair: reading R1            */
            continue;
        double r2 = dx * dx + dy * dy + dz * dz + eps2; /* r_ij^2 + eps^2 */
        double r1i = 1.0 / sqrt(r2);                  /* 1/sqrt(r2) */
        double r2i = r1i * r1i;
        double r3i = r2i * r1i;
        double mr3i = mj[j] * r3i;
        ax += mr3i * dx;                              /* OUTPUT[0..2] += mr3i * d */
        ay += mr3i * dy;
        az += mr3i * dz;
        phi -= mj[j] * r1i;                           /* OUTPUT[6] -= pot */
    }
    out4[0] = ax; out4[1] = ay; out4[2] = az; out4[3] = phi;
}

/*
 * Double-precision inputs.  x_i [n_i][3], x_j [n_j][3], m_j [n_j]; acc [n_i][3]; pot [n_i] or NULL.
 * x_i may alias x_j.  Returns 0, or 1 on a bad argument.
 */
int oracle_force_f64(int64_t n_i, const double *x_i, int64_t n_j, const double *x_j, const double *m_j,
                     double eps2, double *acc, double *pot)
{
    if (n_i < 0 || n_j < 0 || !(eps2 >= 0.0)) return 1;
    if (n_i > 0 && (!x_i || !acc)) return 1;
    if (n_j > 0 && (!x_j || !m_j)) return 1;
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n_i; ++i) {
        double out[4];
        one_i(&x_i[3 * i], n_j, x_j, m_j, eps2, out);
        acc[3 * i + 0] = out[0];
        acc[3 * i + 1] = out[1];
        acc[3 * i + 2] = out[2];
        if (pot) pot[i] = out[3];
    }
    return 0;
}

/*
 * FP32 inputs, each value converted exactly to double (the parity entry: the CUDA path receives
 * the very same FP32 arrays, so input rounding never enters the comparison).  Outputs are double.
 */
int oracle_force_f32(int64_t n_i, const float *x_i, int64_t n_j, const float *x_j, const float *m_j,
                     float eps2, double *acc, double *pot)
{
    if (n_i < 0 || n_j < 0 || !(eps2 >= 0.0f)) return 1;
    if (n_i > 0 && (!x_i || !acc)) return 1;
    if (n_j > 0 && (!x_j || !m_j)) return 1;
    double *xj = (double *)malloc(sizeof(double) * 3 * (size_t)(n_j > 0 ? n_j : 1));
    double *mj = (double *)malloc(sizeof(double) * (size_t)(n_j > 0 ? n_j : 1));
    if (!xj || !mj) { free(xj); free(mj); return 2; }
    for (int64_t j = 0; j < n_j; ++j) {
        xj[3 * j + 0] = (double)x_j[3 * j + 0];
        xj[3 * j + 1] = (double)x_j[3 * j + 1];
        xj[3 * j + 2] = (double)x_j[3 * j + 2];
        mj[j] = (double)m_j[j];
    }
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n_i; ++i) {
        double xi[3] = { (double)x_i[3 * i + 0], (double)x_i[3 * i + 1], (double)x_i[3 * i + 2] };
        double out[4];
        one_i(xi, n_j, xj, mj, (double)eps2, out);
        acc[3 * i + 0] = out[0];
        acc[3 * i + 1] = out[1];
        acc[3 * i + 2] = out[2];
        if (pot) pot[i] = out[3];
    }
    free(xj); free(mj);
    return 0;
}

/*
 * Total energy of a self-gravitating set: E = T + W, T = 1/2 sum m_i |v_i|^2,
 * W = 1/2 sum m_i phi_i with the masked phi above (no self-energy).  FP32 state in (the GPU's own
 * x, v at some step), double arithmetic.  out3 = (T, W, E).
 */
int oracle_energy_f32(int64_t n, const float *x, const float *v, const float *m, float eps2, double out3[3])
{
    if (n < 0 || !out3) return 1;
    double *acc = (double *)malloc(sizeof(double) * 3 * (size_t)(n > 0 ? n : 1));
    double *pot = (double *)malloc(sizeof(double) * (size_t)(n > 0 ? n : 1));
    if (!acc || !pot) { free(acc); free(pot); return 2; }
    int rc = oracle_force_f32(n, x, n, x, m, eps2, acc, pot);
    double T = 0.0, W = 0.0;
    if (rc == 0) {
        for (int64_t i = 0; i < n; ++i) {
            double vx = (double)v[3 * i], vy = (double)v[3 * i + 1], vz = (double)v[3 * i + 2];
            T += 0.5 * (double)m[i] * (vx * vx + vy * vy + vz * vz);
            W += 0.5 * (double)m[i] * pot[i];
        }
        out3[0] = T; out3[1] = W; out3[2] = T + W;
    }
    free(acc); free(pot);
    return rc;
}

/*
 * Kick-drift-kick leapfrog in double precision, state updated in place.
 * x, v [n][3]; m [n]; acc [n][3] and pot [n] receive a and phi at the final time.
 */
int oracle_leapfrog_kdk_f64(int64_t n, double *x, double *v, const double *m, double eps2, double dt,
                            int64_t n_steps, double *acc, double *pot)
{
    if (n < 0 || n_steps < 0 || !(eps2 >= 0.0)) return 1;
    if (n > 0 && (!x || !v || !m || !acc || !pot)) return 1;
    int rc = oracle_force_f64(n, x, n, x, m, eps2, acc, pot);       /* a0 = force(x0) */
    for (int64_t s = 0; s < n_steps && rc == 0; ++s) {
        for (int64_t k = 0; k < 3 * n; ++k) v[k] += acc[k] * (0.5 * dt);   /* kick  dt/2 */
        for (int64_t k = 0; k < 3 * n; ++k) x[k] += v[k] * dt;             /* drift dt   */
        rc = oracle_force_f64(n, x, n, x, m, eps2, acc, pot);              /* a = force(x) */
        for (int64_t k = 0; k < 3 * n; ++k) v[k] += acc[k] * (0.5 * dt);   /* kick  dt/2 */
    }
    return rc;
}

/* ------------------------------------------------------------------------------------------------
 * Row f1: force + jerk + potential for the 4th-order Hermite scheme,
 * the paper's second pipeline description (Fig. A.2, Fig. A.4):
 *
 *     a_i    =  sum_j m_j d / r^3                                   d = r_j - r_i, r^2 = d.d + eps^2
 *     jerk_i =  sum_j m_j [ dv / r^3  -  3 (d.dv) d / r^5 ]         dv = v_j - v_i   (= d a_i / dt)
 *     phi_i  = -sum_j m_j / r
 *
 * Per-pair statements in the order of Fig. A.4: r1i, r2i, r3i, r5i,
 * mr5i = mj r5i, mf = mr5i r2 (= mj r3i), pot = mf r2 (= mj r1i),
 * fx = mf d, jk1 = mf dv, xv = d*dv per component,
 * mf3a = 3 mr5i (xv0+xv1+xv2), jk2 = mf3a d, jk = jk1 - jk2,
 * OUTPUT[0..2] += fx, OUTPUT[3..5] += jk, OUTPUT[6] -= pot.
 * Coincident pairs (all three POSITION differences exactly zero) are skipped (reading R1), whatever
 * their velocities.  Pins (tests/test_oracle_hermite_pins.py): exact two-body rationals, central
 * finite difference of the (separately pinned) acceleration along the flow, exact rational brute
 * force at N <= 6, momentum antisymmetry, Galilean and rotation invariance, circular binary.
 * out7 = (ax, ay, az, jx, jy, jz, phi).
 */
static void one_i_jerk(const double xi[3], const double vi[3], int64_t n_j, const double *xj, const double *vj,
                       const double *mj, double eps2, double out7[7])
{
    double ax = 0.0, ay = 0.0, az = 0.0, jx = 0.0, jy = 0.0, jz = 0.0, phi = 0.0;
    for (int64_t j = 0; j < n_j; ++j) {
        double dx0 = xj[3 * j + 0] - xi[0];            /* dx = xj - xi */
        double dx1 = xj[3 * j + 1] - xi[1];
        double dx2 = xj[3 * j + 2] - xi[2];
        if (dx0 == 0.0 && dx1 == 0.0 && dx2 == 0.0)    /* coincident pair: reading R1 */
            continue;
        double r2 = dx0 * dx0 + dx1 * dx1 + dx2 * dx2 + eps2;
        double r1i = 1.0 / sqrt(r2);
        double r2i = r1i * r1i;
        double r3i = r1i * r2i;
        double r5i = r2i * r3i;
        double mr5i = mj[j] * r5i;
        double mf = mr5i * r2;                         /* = mj / r^3 */
        double pot = mf * r2;                          /* = mj / r */
        double dv0 = vj[3 * j + 0] - vi[0];            /* dv = vj - vi */
        double dv1 = vj[3 * j + 1] - vi[1];
        double dv2 = vj[3 * j + 2] - vi[2];
        double mf3a = 3.0 * mr5i * (dx0 * dv0 + dx1 * dv1 + dx2 * dv2);
        ax += mf * dx0;                                /* OUTPUT[0..2] += fx */
        ay += mf * dx1;
        az += mf * dx2;
        jx += mf * dv0 - mf3a * dx0;                   /* OUTPUT[3..5] += jk1 - jk2 PAPER.md:532-550 */
        jy += mf * dv1 - mf3a * dx1;
        jz += mf * dv2 - mf3a * dx2;
        phi -= pot;                                    /* OUTPUT[6] -= pot */
    }
    out7[0] = ax; out7[1] = ay; out7[2] = az; out7[3] = jx; out7[4] = jy; out7[5] = jz; out7[6] = phi;
}

/* Double inputs.  x_i, v_i [n_i][3]; x_j, v_j [n_j][3]; m_j [n_j]; acc, jerk [n_i][3]; pot [n_i] or NULL. */
int oracle_force_jerk_f64(int64_t n_i, const double *x_i, const double *v_i, int64_t n_j, const double *x_j,
                          const double *v_j, const double *m_j, double eps2, double *acc, double *jerk, double *pot)
{
    if (n_i < 0 || n_j < 0 || !(eps2 >= 0.0)) return 1;
    if (n_i > 0 && (!x_i || !v_i || !acc || !jerk)) return 1;
    if (n_j > 0 && (!x_j || !v_j || !m_j)) return 1;
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n_i; ++i) {
        double out[7];
        one_i_jerk(&x_i[3 * i], &v_i[3 * i], n_j, x_j, v_j, m_j, eps2, out);
        for (int c = 0; c < 3; ++c) { acc[3 * i + c] = out[c]; jerk[3 * i + c] = out[3 + c]; }
        if (pot) pot[i] = out[6];
    }
    return 0;
}

/* FP32 inputs promoted exactly to double (the parity entry); outputs double. */
int oracle_force_jerk_f32(int64_t n_i, const float *x_i, const float *v_i, int64_t n_j, const float *x_j,
                          const float *v_j, const float *m_j, float eps2, double *acc, double *jerk, double *pot)
{
    if (n_i < 0 || n_j < 0 || !(eps2 >= 0.0f)) return 1;
    if (n_i > 0 && (!x_i || !v_i || !acc || !jerk)) return 1;
    if (n_j > 0 && (!x_j || !v_j || !m_j)) return 1;
    size_t nj = (size_t)(n_j > 0 ? n_j : 1);
    double *xj = (double *)malloc(sizeof(double) * 3 * nj);
    double *vj = (double *)malloc(sizeof(double) * 3 * nj);
    double *mj = (double *)malloc(sizeof(double) * nj);
    if (!xj || !vj || !mj) { free(xj); free(vj); free(mj); return 2; }
    for (int64_t k = 0; k < 3 * n_j; ++k) { xj[k] = (double)x_j[k]; vj[k] = (double)v_j[k]; }
    for (int64_t j = 0; j < n_j; ++j) mj[j] = (double)m_j[j];
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n_i; ++i) {
        double xi[3] = { (double)x_i[3 * i + 0], (double)x_i[3 * i + 1], (double)x_i[3 * i + 2] };
        double vi[3] = { (double)v_i[3 * i + 0], (double)v_i[3 * i + 1], (double)v_i[3 * i + 2] };
        double out[7];
        one_i_jerk(xi, vi, n_j, xj, vj, mj, (double)eps2, out);
        for (int c = 0; c < 3; ++c) { acc[3 * i + c] = out[c]; jerk[3 * i + c] = out[3 + c]; }
        if (pot) pot[i] = out[6];
    }
    free(xj); free(vj); free(mj);
    return 0;
}

/* ------------------------------------------------------------------------------------------------
 * Row f3: the softening travels PER i-PARTICLE, as in the paper's own driver,
 * where slot 3 of every i-record is eps2 (Fig. A.1: p_xi[i][3] = eps2;
 * Fig. A.3: eps2 = INPUT_I[3]).  Same sum as one_i() with eps2 -> eps2_i[i].
 * Pins (tests/test_oracle_pins.py, "f3"): a constant array reproduces oracle_force_f64 bit for bit;
 * exact two-body rationals with a different eps2 per i; mpmath brute force.
 */
int oracle_force_eps_i_f64(int64_t n_i, const double *x_i, const double *eps2_i, int64_t n_j, const double *x_j,
                           const double *m_j, double *acc, double *pot)
{
    if (n_i < 0 || n_j < 0) return 1;
    if (n_i > 0 && (!x_i || !eps2_i || !acc)) return 1;
    if (n_j > 0 && (!x_j || !m_j)) return 1;
    for (int64_t i = 0; i < n_i; ++i)
        if (!(eps2_i[i] >= 0.0)) return 1;
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n_i; ++i) {
        double out[4];
        one_i(&x_i[3 * i], n_j, x_j, m_j, eps2_i[i], out);     /* eps2 = INPUT_I[3] */
        acc[3 * i + 0] = out[0];
        acc[3 * i + 1] = out[1];
        acc[3 * i + 2] = out[2];
        if (pot) pot[i] = out[3];
    }
    return 0;
}

/* ------------------------------------------------------------------------------------------------
 * Fourth-order Hermite integration with a shared, constant time step -- the scheme the paper names as the user
 * of its force + jerk pipeline ("Hermite scheme"), not described in the paper itself.
 * Textbook predict - evaluate - correct form (Makino & Aarseth 1992), one evaluation per step:
 *
 *     a0, j0 = force_jerk(x, v)                                   once, before the first step
 *     xp = x + v dt + a0 dt^2/2 + j0 dt^3/6      vp = v + a0 dt + j0 dt^2/2            (predict)
 *     a1, j1 = force_jerk(xp, vp)                                                       (evaluate)
 *     v' = v + (a0 + a1) dt/2 + (j0 - j1) dt^2/12                                       (correct)
 *     x' = x + (v + v') dt/2 + (a0 - a1) dt^2/12
 *     a0, j0 <- a1, j1            (the values at the predicted state are carried to the next step)
 *
 * Pins (tests/test_oracle_hermite_pins.py, "h7"): agreement with an adaptive high-order ODE solver (scipy DOP853)
 * on a three-body problem, error ratio ~16 when dt halves (4th order), energy error far below the leapfrog's.
 * x, v [n][3] updated in place; acc, jerk [n][3] and pot [n] receive the values carried out of the last step.
 */
int oracle_hermite4_f64(int64_t n, double *x, double *v, const double *m, double eps2, double dt, int64_t n_steps,
                        double *acc, double *jerk, double *pot)
{
    if (n < 0 || n_steps < 0 || !(eps2 >= 0.0)) return 1;
    if (n > 0 && (!x || !v || !m || !acc || !jerk || !pot)) return 1;
    size_t n3 = 3 * (size_t)(n > 0 ? n : 1);
    double *xp = (double *)malloc(sizeof(double) * n3), *vp = (double *)malloc(sizeof(double) * n3);
    double *a1 = (double *)malloc(sizeof(double) * n3), *j1 = (double *)malloc(sizeof(double) * n3);
    if (!xp || !vp || !a1 || !j1) { free(xp); free(vp); free(a1); free(j1); return 2; }
    int rc = oracle_force_jerk_f64(n, x, v, n, x, v, m, eps2, acc, jerk, pot);
    const double h = dt, h2 = dt * dt, h3 = dt * dt * dt;
    for (int64_t s = 0; s < n_steps && rc == 0; ++s) {
        for (int64_t k = 0; k < 3 * n; ++k) {                                   /* predict */
            xp[k] = x[k] + v[k] * h + acc[k] * (h2 / 2.0) + jerk[k] * (h3 / 6.0);
            vp[k] = v[k] + acc[k] * h + jerk[k] * (h2 / 2.0);
        }
        rc = oracle_force_jerk_f64(n, xp, vp, n, xp, vp, m, eps2, a1, j1, pot);   /* evaluate */
        for (int64_t k = 0; k < 3 * n; ++k) {                                   /* correct */
            double vn = v[k] + (acc[k] + a1[k]) * (h / 2.0) + (jerk[k] - j1[k]) * (h2 / 12.0);
            x[k] = x[k] + (v[k] + vn) * (h / 2.0) + (acc[k] - a1[k]) * (h2 / 12.0);
            v[k] = vn;
            acc[k] = a1[k];
            jerk[k] = j1[k];
        }
    }
    free(xp); free(vp); free(a1); free(j1);
    return rc;
}

/* ------------------------------------------------------------------------------------------------
 * Row f4, second half: one block step of the 4th-order Hermite scheme with individual (block) time steps -- the
 * "active-subset" use BASELINE.json configs[2] is shaped for (i-set = the particles due now, j-set = everybody).
 * Not in the paper (it only names the Hermite scheme); reading R20 takes the textbook
 * form (Makino 1991; Makino & Aarseth 1992).  Every particle k holds (x, v, a, j) at its OWN time t[k] <= t_now.
 *
 *     for every particle k:   h = t_now - t[k]                                    (predict everybody to t_now)
 *         xp = x + v h + a h^2/2 + j h^3/6        vp = v + a h + j h^2/2
 *     for the active particles i only:
 *         a1, j1 = force_jerk(i-set = (xp, vp) of the active, j-set = (xp, vp, m) of all)            (evaluate)
 *         h = t_now - t[i]
 *         v' = v + (a + a1) h/2 + (j - j1) h^2/12       x' = x + (v + v') h/2 + (a - a1) h^2/12      (correct)
 *         x, v, a, j, t <- x', v', a1, j1, t_now
 *     the others are left exactly as they were (their predicted state is discarded).
 *
 * Who is active and the next step of each particle are the caller's business (the scheduler is outside this call).
 * active[] holds n_act distinct indices in [0, n).  With every particle active and all t equal this is one step of
 * oracle_hermite4_f64.
 * Pins (tests/test_oracle_hermite_pins.py, "h8"): that reduction; inactive particles bitwise untouched; a two-level
 * schedule against scipy DOP853 with 4th-order convergence (fails when stale particles are not predicted or are
 * predicted over the wrong interval); a pure-Python restatement with math.fsum on a tiny case.
 */
int oracle_hermite4_block_step_f64(int64_t n, double *x, double *v, const double *m, double *acc, double *jerk, double *t,
                                   int64_t n_act, const int32_t *active, double t_now, double eps2)
{
    if (n < 0 || n_act < 0 || n_act > n || !(eps2 >= 0.0)) return 1;
    if (n > 0 && (!x || !v || !m || !acc || !jerk || !t)) return 1;
    if (n_act > 0 && !active) return 1;
    for (int64_t q = 0; q < n_act; ++q) if (active[q] < 0 || active[q] >= n) return 1;
    if (n_act == 0) return 0;
    size_t n3 = 3 * (size_t)n, a3 = 3 * (size_t)n_act;
    double *xp = (double *)malloc(sizeof(double) * n3), *vp = (double *)malloc(sizeof(double) * n3);
    double *xi = (double *)malloc(sizeof(double) * a3), *vi = (double *)malloc(sizeof(double) * a3);
    double *a1 = (double *)malloc(sizeof(double) * a3), *j1 = (double *)malloc(sizeof(double) * a3);
    if (!xp || !vp || !xi || !vi || !a1 || !j1) { free(xp); free(vp); free(xi); free(vi); free(a1); free(j1); return 2; }
    for (int64_t k = 0; k < n; ++k) {                                           /* predict everybody */
        const double h = t_now - t[k], h2 = h * h, h3 = h * h * h;
        for (int c = 0; c < 3; ++c) {
            const size_t e = 3 * (size_t)k + c;
            xp[e] = x[e] + v[e] * h + acc[e] * (h2 / 2.0) + jerk[e] * (h3 / 6.0);
            vp[e] = v[e] + acc[e] * h + jerk[e] * (h2 / 2.0);
        }
    }
    for (int64_t q = 0; q < n_act; ++q)                                         /* the i-set: the active, predicted */
        for (int c = 0; c < 3; ++c) {
            xi[3 * q + c] = xp[3 * (size_t)active[q] + c];
            vi[3 * q + c] = vp[3 * (size_t)active[q] + c];
        }
    int rc = oracle_force_jerk_f64(n_act, xi, vi, n, xp, vp, m, eps2, a1, j1, NULL);   /* evaluate */
    for (int64_t q = 0; q < n_act && rc == 0; ++q) {                            /* correct the active */
        const size_t k = (size_t)active[q];
        const double h = t_now - t[k], h2 = h * h;
        for (int c = 0; c < 3; ++c) {
            const size_t e = 3 * k + c;
            const double vn = v[e] + (acc[e] + a1[3 * q + c]) * (h / 2.0) + (jerk[e] - j1[3 * q + c]) * (h2 / 12.0);
            x[e] = x[e] + (v[e] + vn) * (h / 2.0) + (acc[e] - a1[3 * q + c]) * (h2 / 12.0);
            v[e] = vn;
            acc[e] = a1[3 * q + c];
            jerk[e] = j1[3 * q + c];
        }
        t[k] = t_now;
    }
    free(xp); free(vp); free(xi); free(vi); free(a1); free(j1);
    return rc;
}

/* ------------------------------------------------------------------------------------------------
 * Row f3, a central force other than gravity: the paper lists "van der Waals molecular interactions" among the
 * interactions its generalised library runs (section 4.5) and gives no formula; reading R19
 * takes the textbook 12-6 Lennard-Jones pair with Lorentz-Berthelot mixing, all pairs, no cut-off:
 *
 *     i-record (x, y, z, sigma_i / 2, sqrt(eps_i))      j-record (x, y, z, sigma_j / 2, sqrt(eps_j))
 *     sigma = sigma_i / 2 + sigma_j / 2       eps = sqrt(eps_i) sqrt(eps_j)       d = r_j - r_i      r2 = d . d
 *     s6 = (sigma^2 / r2)^3
 *     F_i = - sum_j 24 eps (2 s6^2 - s6) / r2 * d            (force ON i: repulsive inside r = 2^(1/6) sigma)
 *     U_i =   sum_j  4 eps (s6^2 - s6)                       (pair energies seen by i; E_total = 1/2 sum_i U_i)
 *
 * A pair with d = 0 contributes nothing (reading R1).  Result record (Fx, Fy, Fz, U), plain double sums in j order.
 * Pins (tests/test_oracle_pins.py, "lj"): zero force and U = -eps at r = 2^(1/6) sigma; U = 0 and |F| = 24 eps / sigma
 * at r = sigma; exact rationals at r = 2 sigma; the mixing rule against a single-species pair; Newton's third law;
 * F = -grad E_total by central differences; a pure-Python double loop.
 */
int oracle_lj_f64(int64_t n_i, const double *p_xi, int64_t n_j, const double *p_xj, double *p_fi)
{
    if (n_i < 0 || n_j < 0) return 1;
    if (n_i > 0 && (!p_xi || !p_fi)) return 1;
    if (n_j > 0 && !p_xj) return 1;
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n_i; ++i) {
        const double *I = &p_xi[5 * i];
        double fx = 0.0, fy = 0.0, fz = 0.0, u = 0.0;
        for (int64_t j = 0; j < n_j; ++j) {
            const double *J = &p_xj[5 * j];
            const double dx = J[0] - I[0], dy = J[1] - I[1], dz = J[2] - I[2];
            const double r2 = dx * dx + dy * dy + dz * dz;
            if (r2 == 0.0) continue;                                   /* coincident pair: nothing (R1) */
            const double sigma = I[3] + J[3], eps = I[4] * J[4];
            const double s2 = sigma * sigma / r2, s6 = s2 * s2 * s2;
            const double f = 24.0 * eps * (2.0 * s6 * s6 - s6) / r2;
            fx -= f * dx;
            fy -= f * dy;
            fz -= f * dz;
            u += 4.0 * eps * (s6 * s6 - s6);
        }
        p_fi[4 * i + 0] = fx;
        p_fi[4 * i + 1] = fy;
        p_fi[4 * i + 2] = fz;
        p_fi[4 * i + 3] = u;
    }
    return 0;
}
