/* ORACLE -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, fp64 CPU implementation of what the index-based multi-walk force path computes
 * (arXiv 1907.02290, /root/reference/PAPER.md; "P:n" = line n of that file).  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call it.  It
 * shares no code with the CUDA library (paper_1907_02290_b200/csrc) and is never tuned.
 *
 * What it evaluates:
 *   orc_monopoles  P:160, P:848  monopole (centre-of-mass) moment of every tree cell, bottom line
 *                  of the definition: M_c = sum m_p, X_c = sum m_p x_p / M_c over the cell's
 *                  particle range.  Kept in fp64 (never rounded to fp32).
 *   orc_forces     P:77, P:181, P:441-477  for each i-group, each particle i of the group: the
 *                  softened Newtonian sum over the group's shared interaction list -- EPJ entries
 *                  are particle indices, SPJ entries are cell indices whose (X_c, M_c) act as one
 *                  particle ("a SPJ represents a node of Barnes-Hut tree", P:387 same kernel).
 *                  acc_i = G sum_k m_k d / (|d|^2 + eps^2)^(3/2),  d = x_k - x_i
 *                  pot_i = -G sum_k m_k / (|d|^2 + eps^2)^(1/2)
 *                  The paper never prints the formula; it gives eps2 = eps*eps, the
 *                  float4 (x,y,z,m) -> (ax,ay,az,pot) layout and "monopole"
 *                  (P:197).  Readings S1-S5 in DESIGN.md: Plummer softening, the same eps
 *                  for EPJ and SPJ, the entry whose INDEX equals i is skipped (a different particle
 *                  at the same position is a real pair), pot <= 0 and includes G.
 *   orc_direct     the plain O(N^2) definition of the same sum over all other particles.
 *   orc_quadrupoles, orc_forces_quad   (the paper says "multipole moments", and
 *                  measures the monopole case only)  second moment of every cell about its centre of mass,
 *                  Q_c = sum m_p (x_p - X_c)(x_p - X_c)^T, and the list evaluation in which an SPJ entry acts
 *                  through M_c and Q_c: the Taylor expansion to second order in (x_p - X_c) of the SAME softened
 *                  kernel (reading S22 in DESIGN.md), with R = X_c - x_i, s^2 = |R|^2 + eps^2:
 *                    pot_i -= G [ M/s - tr(Q)/(2 s^3) + 3 (R.Q.R)/(2 s^5) ]
 *                    acc_i += G [ M R/s^3 - 3 tr(Q) R/(2 s^5) - 3 (Q R)/s^5 + 15 (R.Q.R) R/(2 s^7) ]
 *                  EPJ entries are evaluated exactly as in orc_forces.
 *   orc_kick_drift, orc_kick   the kick-drift-kick leapfrog BASELINE.json's config 5 names (the orbit
 *                  integration is step 5 of the paper's procedure; section 7.3, P:1171-1185,
 *                  proposes moving it to the accelerator): v += a dt/2, x += v dt; and v += a dt/2.
 *                  In fp64 from fp32 inputs (reading S14b in DESIGN.md).
 *
 * Inputs are the fp32 particle array exactly as uploaded to the GPU; every value is widened to
 * double before any arithmetic.  OpenMP only distributes groups / particles over threads; each
 * sum runs in list order.  No blocking, no SIMD intrinsics, no reordering.
 */
#include <math.h>
#include <stdint.h>
#ifdef _OPENMP
#include <omp.h>
#endif

int orc_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void orc_set_num_threads(int n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* mom[4*c + 0..2] = X_c, mom[4*c + 3] = M_c.  cells4 = (first_ptcl, n_ptcl, first_child, n_child). */
void orc_monopoles(int64_t n_cell, const int32_t* cells4, const float* posm, double* mom) {
    int64_t c;
#pragma omp parallel for schedule(dynamic, 64)
    for (c = 0; c < n_cell; ++c) {
        int64_t first = cells4[4 * c + 0], cnt = cells4[4 * c + 1];
        double m = 0.0, sx = 0.0, sy = 0.0, sz = 0.0;
        for (int64_t p = first; p < first + cnt; ++p) {
            double mp = (double)posm[4 * p + 3];
            m += mp;
            sx += mp * (double)posm[4 * p + 0];
            sy += mp * (double)posm[4 * p + 1];
            sz += mp * (double)posm[4 * p + 2];
        }
        mom[4 * c + 0] = sx / m;
        mom[4 * c + 1] = sy / m;
        mom[4 * c + 2] = sz / m;
        mom[4 * c + 3] = m;
    }
}

static void pair_term(double xi, double yi, double zi, double xk, double yk, double zk, double mk, double eps2,
                      double* ax, double* ay, double* az, double* pot) {
    double dx = xk - xi, dy = yk - yi, dz = zk - zi;
    double r2 = dx * dx + dy * dy + dz * dz + eps2;
    double rinv = 1.0 / sqrt(r2);
    double mr3 = mk * rinv * rinv * rinv;
    *ax += mr3 * dx;
    *ay += mr3 * dy;
    *az += mr3 * dz;
    *pot -= mk * rinv;
}

/* Evaluates groups sel[0..n_sel) (or all groups 0..n_sel-1 when sel == NULL).
 * acc: 3 doubles per particle, pot: 1 per particle, indexed by tree-order particle position; only the
 * selected groups' particles are written.  mom comes from orc_monopoles on the SAME posm. */
void orc_forces(int64_t n_sel, const int64_t* sel, const int32_t* grp_first, const int32_t* grp_n,
                const int64_t* epj_off, const int32_t* epj_id, const int64_t* spj_off, const int32_t* spj_id,
                const float* posm, const double* mom, double eps, double G, double* acc, double* pot) {
    const double eps2 = eps * eps;
    int64_t s;
#pragma omp parallel for schedule(dynamic, 1)
    for (s = 0; s < n_sel; ++s) {
        int64_t g = sel ? sel[s] : s;
        int64_t first = grp_first[g], cnt = grp_n[g];
        for (int64_t i = first; i < first + cnt; ++i) {
            double xi = (double)posm[4 * i + 0], yi = (double)posm[4 * i + 1], zi = (double)posm[4 * i + 2];
            double ax = 0.0, ay = 0.0, az = 0.0, p = 0.0;
            for (int64_t e = epj_off[g]; e < epj_off[g + 1]; ++e) {
                int64_t k = epj_id[e];
                if (k == i) continue;
                pair_term(xi, yi, zi, (double)posm[4 * k + 0], (double)posm[4 * k + 1], (double)posm[4 * k + 2],
                          (double)posm[4 * k + 3], eps2, &ax, &ay, &az, &p);
            }
            for (int64_t e = spj_off[g]; e < spj_off[g + 1]; ++e) {
                int64_t c = spj_id[e];
                pair_term(xi, yi, zi, mom[4 * c + 0], mom[4 * c + 1], mom[4 * c + 2], mom[4 * c + 3], eps2, &ax, &ay, &az, &p);
            }
            acc[3 * i + 0] = G * ax;
            acc[3 * i + 1] = G * ay;
            acc[3 * i + 2] = G * az;
            pot[i] = G * p;
        }
    }
}

/* quad[6*c + 0..5] = (Qxx, Qyy, Qzz, Qxy, Qxz, Qyz) of cell c about its centre of mass mom[4*c + 0..2], straight
 * from the definition over the cell's particle range. */
void orc_quadrupoles(int64_t n_cell, const int32_t* cells4, const float* posm, const double* mom, double* quad) {
    int64_t c;
#pragma omp parallel for schedule(dynamic, 64)
    for (c = 0; c < n_cell; ++c) {
        int64_t first = cells4[4 * c + 0], cnt = cells4[4 * c + 1];
        double q[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
        for (int64_t p = first; p < first + cnt; ++p) {
            double mp = (double)posm[4 * p + 3];
            double yx = (double)posm[4 * p + 0] - mom[4 * c + 0];
            double yy = (double)posm[4 * p + 1] - mom[4 * c + 1];
            double yz = (double)posm[4 * p + 2] - mom[4 * c + 2];
            q[0] += mp * yx * yx;
            q[1] += mp * yy * yy;
            q[2] += mp * yz * yz;
            q[3] += mp * yx * yy;
            q[4] += mp * yx * yz;
            q[5] += mp * yy * yz;
        }
        for (int k = 0; k < 6; ++k) quad[6 * c + k] = q[k];
    }
}

/* Monopole + quadrupole term of one cell on particle i (see the header). */
static void cell_term_quad(double xi, double yi, double zi, const double* X, double M, const double* Q, double eps2,
                           double* ax, double* ay, double* az, double* pot) {
    double Rx = X[0] - xi, Ry = X[1] - yi, Rz = X[2] - zi;
    double s2 = Rx * Rx + Ry * Ry + Rz * Rz + eps2;
    double s1 = sqrt(s2);
    double s3 = s2 * s1, s5 = s3 * s2, s7 = s5 * s2;
    double tr = Q[0] + Q[1] + Q[2];
    double QRx = Q[0] * Rx + Q[3] * Ry + Q[4] * Rz;
    double QRy = Q[3] * Rx + Q[1] * Ry + Q[5] * Rz;
    double QRz = Q[4] * Rx + Q[5] * Ry + Q[2] * Rz;
    double RQR = Rx * QRx + Ry * QRy + Rz * QRz;
    *pot -= M / s1 - tr / (2.0 * s3) + 3.0 * RQR / (2.0 * s5);
    double cR = M / s3 - 3.0 * tr / (2.0 * s5) + 15.0 * RQR / (2.0 * s7);
    *ax += cR * Rx - 3.0 * QRx / s5;
    *ay += cR * Ry - 3.0 * QRy / s5;
    *az += cR * Rz - 3.0 * QRz / s5;
}

/* As orc_forces, with SPJ entries acting through monopole and quadrupole (quad from orc_quadrupoles). */
void orc_forces_quad(int64_t n_sel, const int64_t* sel, const int32_t* grp_first, const int32_t* grp_n,
                     const int64_t* epj_off, const int32_t* epj_id, const int64_t* spj_off, const int32_t* spj_id,
                     const float* posm, const double* mom, const double* quad, double eps, double G, double* acc, double* pot) {
    const double eps2 = eps * eps;
    int64_t s;
#pragma omp parallel for schedule(dynamic, 1)
    for (s = 0; s < n_sel; ++s) {
        int64_t g = sel ? sel[s] : s;
        int64_t first = grp_first[g], cnt = grp_n[g];
        for (int64_t i = first; i < first + cnt; ++i) {
            double xi = (double)posm[4 * i + 0], yi = (double)posm[4 * i + 1], zi = (double)posm[4 * i + 2];
            double ax = 0.0, ay = 0.0, az = 0.0, p = 0.0;
            for (int64_t e = epj_off[g]; e < epj_off[g + 1]; ++e) {
                int64_t k = epj_id[e];
                if (k == i) continue;
                pair_term(xi, yi, zi, (double)posm[4 * k + 0], (double)posm[4 * k + 1], (double)posm[4 * k + 2],
                          (double)posm[4 * k + 3], eps2, &ax, &ay, &az, &p);
            }
            for (int64_t e = spj_off[g]; e < spj_off[g + 1]; ++e) {
                int64_t c = spj_id[e];
                cell_term_quad(xi, yi, zi, mom + 4 * c, mom[4 * c + 3], quad + 6 * c, eps2, &ax, &ay, &az, &p);
            }
            acc[3 * i + 0] = G * ax;
            acc[3 * i + 1] = G * ay;
            acc[3 * i + 2] = G * az;
            pot[i] = G * p;
        }
    }
}

/* Direct summation over all other particles (the definition Barnes-Hut approximates). */
void orc_direct(int64_t n, const float* posm, double eps, double G, double* acc, double* pot) {
    const double eps2 = eps * eps;
    int64_t i;
#pragma omp parallel for schedule(static)
    for (i = 0; i < n; ++i) {
        double xi = (double)posm[4 * i + 0], yi = (double)posm[4 * i + 1], zi = (double)posm[4 * i + 2];
        double ax = 0.0, ay = 0.0, az = 0.0, p = 0.0;
        for (int64_t k = 0; k < n; ++k) {
            if (k == i) continue;
            pair_term(xi, yi, zi, (double)posm[4 * k + 0], (double)posm[4 * k + 1], (double)posm[4 * k + 2],
                      (double)posm[4 * k + 3], eps2, &ax, &ay, &az, &p);
        }
        acc[3 * i + 0] = G * ax;
        acc[3 * i + 1] = G * ay;
        acc[3 * i + 2] = G * az;
        pot[i] = G * p;
    }
}

/* Kick-drift of the leapfrog: vout = v + a dt/2, xout = x + vout dt.  posm: 4 floats per particle (x,y,z,m);
 * vel4 and accp4: 4 floats per particle (3 used).  Outputs 3 doubles per particle. */
void orc_kick_drift(int64_t n, const float* posm, const float* vel4, const float* accp4, double dt, double* xout, double* vout) {
    for (int64_t i = 0; i < n; ++i)
        for (int d = 0; d < 3; ++d) {
            double v = (double)vel4[4 * i + d] + (double)accp4[4 * i + d] * (0.5 * dt);
            vout[3 * i + d] = v;
            xout[3 * i + d] = (double)posm[4 * i + d] + v * dt;
        }
}

/* Closing half kick: vout = v + a dt/2. */
void orc_kick(int64_t n, const float* vel4, const float* accp4, double dt, double* vout) {
    for (int64_t i = 0; i < n; ++i)
        for (int d = 0; d < 3; ++d) vout[3 * i + d] = (double)vel4[4 * i + d] + (double)accp4[4 * i + d] * (0.5 * dt);
}
