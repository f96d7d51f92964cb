/*
 * nbody_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, obviously-correct FP64 CPU statement of what the hot path computes: the regular-force
 * step of the fourth-order Hermite / Ahmad-Cohen neighbour scheme (arXiv 1504.03687).  It shares no
 * code, header, table or helper with the CUDA path (paper_1504_03687_b200/csrc) and neither side
 * imports the other.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may build, load or call it.
 *
 * The method is exact (a direct sum), so this file is the definition written out -- no blocking,
 * tiling, fusion or reordering; j runs 0..N-1 in order for every i.  Pair terms are evaluated in
 * double; the seven running sums per i are kept in long double (x87 80-bit here) so the oracle's own
 * rounding is far below 1e-12.  OpenMP over i only (each i is independent).
 *
 * Passages followed (P:NNN = /root/reference/PAPER.md line NNN; the paper prints no equation for
 * the force, so the formulas are the textbook Hermite scheme it names -- DESIGN.md "Readings"):
 *   P:45, P:115  Hermite uses the force and its first time derivative, evaluated from PREDICTED
 *                positions and velocities;
 *   P:141        "Pred.": all particles are predicted for the regular force;
 *   P:49         regular force = sum over particles OUTSIDE the neighbour radius;
 *   P:69, P:139  the neighbour list is determined during the regular-force pass; the same library
 *                gives the potential.
 * Pins (tests/test_oracle_pins.py): two-body closed forms, finite-difference jerk = d(acc)/dt and
 * acc = -grad(pot), sum m a = 0, regular + neighbour sum = total, Plummer W = -3 pi/32 GM^2/a,
 * KD-tree neighbour sets, brute force at N <= 64, dyadic-exact predictor.  Nothing is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#ifdef _OPENMP
#include <omp.h>
#endif

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* Hermite predictor, Taylor series to the jerk term (reading R2):
 *   dt = t - t0[j]
 *   xp = x0 + v0 dt + a0 dt^2/2 + j0 dt^3/6
 *   vp = v0 + a0 dt + j0 dt^2/2
 * a0, j0 are the total acceleration and jerk at t0 (not pre-divided). Arrays are [N][3] row-major. */
void orc_predict(int64_t N, const double *x0, const double *v0, const double *a0, const double *j0,
                 const double *t0, double t, double *xp, double *vp)
{
    for (int64_t j = 0; j < N; ++j) {
        double dt = t - t0[j];
        double dt2 = dt * dt;
        double dt3 = dt2 * dt;
        for (int c = 0; c < 3; ++c) {
            int64_t q = 3 * j + c;
            xp[q] = x0[q] + v0[q] * dt + a0[q] * (dt2 / 2.0) + j0[q] * (dt3 / 6.0);
            vp[q] = v0[q] + a0[q] * dt + j0[q] * (dt2 / 2.0);
        }
    }
}

/* Regular force, jerk, potential and neighbour list for a block of active particles
 * (SURVEY.md 8(c) pseudo-code):
 *
 *   for each k:  i = idx_i[k]
 *     for each j != i (by INDEX):  r = xp[j]-xp[i], v = vp[j]-vp[i], r2 = r.r, rv = r.v
 *        if r2 < h2_i[k]:  j is a neighbour: listed, excluded from acc/jerk/pot (kept in *_nb)
 *        else:             acc  += m_j r / r2^(3/2)
 *                          jerk += m_j ( v / r2^(3/2) - 3 rv r / r2^(5/2) )
 *                          pot  -= m_j / r2^(1/2)
 *     nnb[k] = TRUE count; overflow[k] = nnb[k] > cap; nblist[k][0..min(nnb,cap)) ascending j.
 *
 * acc_nb/jerk_nb/pot_nb (may be NULL) receive the same three sums over the NEIGHBOURS, so that
 * regular + neighbour = total can be checked and the alternative reading of `pot` is one add away.
 * nblist may be NULL. Returns 0. */
int orc_regular(int64_t N, const double *m, const double *xp, const double *vp,
                int32_t n_i, const int32_t *idx_i, const double *h2_i, int32_t cap,
                double *acc, double *jerk, double *pot,
                double *acc_nb, double *jerk_nb, double *pot_nb,
                int32_t *nnb, int32_t *nblist, int32_t *overflow)
{
#pragma omp parallel for schedule(dynamic, 4)
    for (int32_t k = 0; k < n_i; ++k) {
        const int64_t i = idx_i[k];
        const double h2 = h2_i[k];
        const double xi = xp[3 * i], yi = xp[3 * i + 1], zi = xp[3 * i + 2];
        const double ui = vp[3 * i], vi = vp[3 * i + 1], wi = vp[3 * i + 2];
        long double A[3] = {0, 0, 0}, J[3] = {0, 0, 0}, P = 0;
        long double An[3] = {0, 0, 0}, Jn[3] = {0, 0, 0}, Pn = 0;
        int64_t count = 0;
        for (int64_t j = 0; j < N; ++j) {
            if (j == i) continue;
            double rx = xp[3 * j] - xi, ry = xp[3 * j + 1] - yi, rz = xp[3 * j + 2] - zi;
            double vx = vp[3 * j] - ui, vy = vp[3 * j + 1] - vi, vz = vp[3 * j + 2] - wi;
            double r2 = rx * rx + ry * ry + rz * rz;
            double rv = rx * vx + ry * vy + rz * vz;
            double r1 = sqrt(r2);
            double mr3 = m[j] / (r2 * r1);              /* m / r^3 */
            double c = 3.0 * rv / r2;                   /* 3 (r.v)/r^2 */
            double ax = mr3 * rx, ay = mr3 * ry, az = mr3 * rz;
            double jx = mr3 * (vx - c * rx), jy = mr3 * (vy - c * ry), jz = mr3 * (vz - c * rz);
            double ph = -m[j] / r1;
            if (r2 < h2) {
                if (nblist && count < cap) nblist[(int64_t)k * cap + count] = (int32_t)j;
                ++count;
                An[0] += ax; An[1] += ay; An[2] += az;
                Jn[0] += jx; Jn[1] += jy; Jn[2] += jz;
                Pn += ph;
            } else {
                A[0] += ax; A[1] += ay; A[2] += az;
                J[0] += jx; J[1] += jy; J[2] += jz;
                P += ph;
            }
        }
        for (int c = 0; c < 3; ++c) {
            acc[3 * k + c] = (double)A[c];
            jerk[3 * k + c] = (double)J[c];
            if (acc_nb) acc_nb[3 * k + c] = (double)An[c];
            if (jerk_nb) jerk_nb[3 * k + c] = (double)Jn[c];
        }
        pot[k] = (double)P;
        if (pot_nb) pot_nb[k] = (double)Pn;
        nnb[k] = (int32_t)count;
        overflow[k] = count > cap ? 1 : 0;
    }
    return 0;
}

/* Boundary-band pairs (BASELINE.json north_star: pairs with |r2-h2|/h2 < band are "reported
 * separately").  For every k and every j != idx_i[k] with h2 > 0 and
 * |r2 - h2| < band * h2, emit (k, j, r2) and the pair's seven terms
 * (acc[3], jerk[3], pot) exactly as orc_regular evaluates them, so that a harness can move a pair
 * whose class the FP32 kernel decided differently to the side the kernel chose.
 * OpenMP over k; the rare appends are serialised, so the output order is unspecified (the Python
 * wrapper sorts by (k, j)).  Returns the number of band pairs found (may exceed max_pairs; only
 * max_pairs of them are stored). */
int64_t orc_band_pairs(int64_t N, const double *m, const double *xp, const double *vp,
                       int32_t n_i, const int32_t *idx_i, const double *h2_i, double band,
                       int64_t max_pairs, int32_t *k_out, int32_t *j_out, double *r2_out,
                       double *terms_out)
{
    int64_t found = 0;
#pragma omp parallel for schedule(dynamic, 4)
    for (int32_t k = 0; k < n_i; ++k) {
        const int64_t i = idx_i[k];
        const double h2 = h2_i[k];
        if (!(h2 > 0.0)) continue;
        const double lo = h2 * (1.0 - band), hi = h2 * (1.0 + band);
        for (int64_t j = 0; j < N; ++j) {
            if (j == i) continue;
            double rx = xp[3 * j] - xp[3 * i], ry = xp[3 * j + 1] - xp[3 * i + 1],
                   rz = xp[3 * j + 2] - xp[3 * i + 2];
            double r2 = rx * rx + ry * ry + rz * rz;
            if (!(r2 > lo && r2 < hi)) continue;
#pragma omp critical(orc_band_append)
            {
            if (found < max_pairs) {
                double vx = vp[3 * j] - vp[3 * i], vy = vp[3 * j + 1] - vp[3 * i + 1],
                       vz = vp[3 * j + 2] - vp[3 * i + 2];
                double rv = rx * vx + ry * vy + rz * vz;
                double r1 = sqrt(r2);
                double mr3 = m[j] / (r2 * r1);
                double c = 3.0 * rv / r2;
                double *T = terms_out + 7 * found;
                T[0] = mr3 * rx; T[1] = mr3 * ry; T[2] = mr3 * rz;
                T[3] = mr3 * (vx - c * rx); T[4] = mr3 * (vy - c * ry); T[5] = mr3 * (vz - c * rz);
                T[6] = -m[j] / r1;
                k_out[found] = k; j_out[found] = (int32_t)j; r2_out[found] = r2;
            }
            ++found;
            }
        }
    }
    return found;
}

/* Neighbour ("irregular") force, jerk and potential ("the irregular
 * force accumulates only the neighbor forces"; "predict all neighbors and do the force
 * calculation within one loop").  For each k, i = idx_i[k]: particle i and every listed
 * j = nblist[k][e], e < min(nnb[k], cap), are predicted to time t with the polynomial of
 * orc_predict (reading R2), then
 *     acc[k]  = sum m_j r / r^3
 *     jerk[k] = sum m_j ( v / r^3 - 3 (r.v) r / r^5 )
 *     pot[k]  = - sum m_j / r            r = xp_j - xp_i, v = vp_j - vp_i
 * over the listed j in list order; pair terms in double, sums in long double.  The state arrays
 * are the caller's [N][3] / [N] inputs at the particles' own times t0.  Returns 0.
 * Pins (tests/test_oracle_pins.py): equals orc_regular's neighbour sums for the lists orc_regular
 * itself emits; regular + irregular = total; numpy brute force; two-body golden values. */
int orc_irregular(int64_t N, const double *m, const double *x0, const double *v0, const double *a0,
                  const double *j0, const double *t0, double t, int32_t n_i, const int32_t *idx_i,
                  const int32_t *nnb, const int32_t *nblist, int32_t cap, double *acc, double *jerk,
                  double *pot)
{
    (void)N;
#pragma omp parallel for schedule(dynamic, 16)
    for (int32_t k = 0; k < n_i; ++k) {
        const int64_t i = idx_i[k];
        double xi[3], vi[3];
        {
            double dt = t - t0[i], dt2 = dt * dt, dt3 = dt2 * dt;
            for (int c = 0; c < 3; ++c) {
                int64_t q = 3 * i + c;
                xi[c] = x0[q] + v0[q] * dt + a0[q] * (dt2 / 2.0) + j0[q] * (dt3 / 6.0);
                vi[c] = v0[q] + a0[q] * dt + j0[q] * (dt2 / 2.0);
            }
        }
        long double A[3] = {0, 0, 0}, J[3] = {0, 0, 0}, P = 0;
        int32_t cnt = nnb[k] < cap ? nnb[k] : cap;
        for (int32_t e = 0; e < cnt; ++e) {
            const int64_t j = nblist[(int64_t)k * cap + e];
            double dt = t - t0[j], dt2 = dt * dt, dt3 = dt2 * dt;
            double r[3], v[3];
            for (int c = 0; c < 3; ++c) {
                int64_t q = 3 * j + c;
                double xj = x0[q] + v0[q] * dt + a0[q] * (dt2 / 2.0) + j0[q] * (dt3 / 6.0);
                double vj = v0[q] + a0[q] * dt + j0[q] * (dt2 / 2.0);
                r[c] = xj - xi[c];
                v[c] = vj - vi[c];
            }
            double r2 = r[0] * r[0] + r[1] * r[1] + r[2] * r[2];
            double rv = r[0] * v[0] + r[1] * v[1] + r[2] * v[2];
            double r1 = sqrt(r2);
            double mr3 = m[j] / (r2 * r1);
            double c3 = 3.0 * rv / r2;
            for (int c = 0; c < 3; ++c) {
                A[c] += mr3 * r[c];
                J[c] += mr3 * (v[c] - c3 * r[c]);
            }
            P -= m[j] / r1;
        }
        for (int c = 0; c < 3; ++c) {
            acc[3 * k + c] = (double)A[c];
            jerk[3 * k + c] = (double)J[c];
        }
        pot[k] = (double)P;
    }
    return 0;
}
