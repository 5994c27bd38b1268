/* ORACLE -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, fp64 CPU implementation of the SHORT-RANGE workload evaluated through the same index lists
 * (arXiv 1907.02290, /root/reference/PAPER.md, "P:n" = line n):
 *   P:79   "In the case of short-range interaction such as SPH interaction between particles, we still use treewalk
 *           but with cell-opening criterion different from the standard opening angle."
 *   P:109-111  a particle record "can be much larger in the case of SPH" -- the reason indices pay off more
 *   P:117  lists of SPH / molecular-dynamics runs can be reused because the time step is stability-limited
 * The paper names the interaction ("SPH") but prints no formula; reading S23 of DESIGN.md takes the textbook
 * form: cubic-spline (M4) kernel of Monaghan & Lattanzio with support 2h in three dimensions,
 *     W(r,h)    = 1/(pi h^3) * { 1 - 3/2 q^2 + 3/4 q^3  (q < 1);  1/4 (2 - q)^3  (1 <= q < 2);  0  (q >= 2) },  q = r/h
 *     dW/dr     = 1/(pi h^4) * { -3 q + 9/4 q^2         (q < 1); -3/4 (2 - q)^2  (1 <= q < 2);  0  (q >= 2) }
 *   orc_sph_density  gather density with the i-particle's own smoothing length, self term included:
 *                    rho_i = sum_{k in list} m_k W(|x_i - x_k|, h_i);  then the ideal-gas quantity
 *                    P_i / rho_i^2 = (gamma - 1) u_i / rho_i
 *   orc_sph_hydro    pressure-gradient acceleration with the symmetrised kernel gradient (momentum conserving):
 *                    a_i = - sum_{k != i} m_k (P_i/rho_i^2 + P_k/rho_k^2) * 1/2 [gradW(r_ik, h_i) + gradW(r_ik, h_k)],
 *                    gradW(r, h) = dW/dr (x_i - x_k)/r ;  a pair at zero distance contributes nothing (dW/dr(0) = 0).
 *                    Also returns scale_i = sum_k |term_k| (the sum of the magnitudes of the terms), the natural unit
 *                    for an absolute error of a sum that cancels.
 *   orc_sph_*_direct the same sums over ALL particles (the kernel has compact support, so a complete neighbour
 *                    list must give exactly these).
 * Only artificial-viscosity-free hydrodynamics is evaluated (no velocity terms).
 *
 * Inputs are fp32 arrays exactly as uploaded to the GPU -- posm (x,y,z,m) and the per-particle record
 * sph4 = (h, u, rho, P/rho^2) -- widened to double before any arithmetic.  OpenMP only distributes groups /
 * particles; each sum runs in list order.  Shares no code with paper_1907_02290_b200/csrc.
 */
#include <math.h>
#include <stdint.h>

static const double ORC_PI = 3.14159265358979323846;

static double sph_w(double r, double h) {
    double q = r / h;
    double s = 1.0 / (ORC_PI * h * h * h);
    if (q < 1.0) return s * (1.0 - 1.5 * q * q + 0.75 * q * q * q);
    if (q < 2.0) return s * 0.25 * (2.0 - q) * (2.0 - q) * (2.0 - q);
    return 0.0;
}

static double sph_dwdr(double r, double h) {
    double q = r / h;
    double s = 1.0 / (ORC_PI * h * h * h * h);
    if (q < 1.0) return s * (-3.0 * q + 2.25 * q * q);
    if (q < 2.0) return s * (-0.75 * (2.0 - q) * (2.0 - q));
    return 0.0;
}

/* test hooks: the kernel and its radial derivative (pinned by quadrature and finite differences) */
double orc_sph_w(double r, double h) { return sph_w(r, h); }
double orc_sph_dwdr(double r, double h) { return sph_dwdr(r, h); }

static double dist(const float* posm, int64_t i, int64_t k) {
    double dx = (double)posm[4 * i + 0] - (double)posm[4 * k + 0];
    double dy = (double)posm[4 * i + 1] - (double)posm[4 * k + 1];
    double dz = (double)posm[4 * i + 2] - (double)posm[4 * k + 2];
    return sqrt(dx * dx + dy * dy + dz * dz);
}

/* rho[i], pr2[i] for the particles of groups sel[0..n_sel) (all groups 0..n_sel-1 when sel == NULL). */
void orc_sph_density(int64_t n_sel, const int64_t* sel, const int32_t* grp_first, const int32_t* grp_n,
                     const int64_t* epj_off, const int32_t* epj_id, const float* posm, const float* sph4, double gamma,
                     double* rho, double* pr2) {
    int64_t s;
#pragma omp parallel for schedule(dynamic, 1)
    for (s = 0; s < n_sel; ++s) {
        int64_t g = sel ? sel[s] : s;
        int64_t first = grp_first[g], cnt = grp_n[g];
        for (int64_t i = first; i < first + cnt; ++i) {
            double hi = (double)sph4[4 * i + 0], ui = (double)sph4[4 * i + 1];
            double sum = 0.0;
            for (int64_t e = epj_off[g]; e < epj_off[g + 1]; ++e) {
                int64_t k = epj_id[e];
                sum += (double)posm[4 * k + 3] * sph_w(dist(posm, i, k), hi);
            }
            rho[i] = sum;
            pr2[i] = (gamma - 1.0) * ui / sum;
        }
    }
}

void orc_sph_density_direct(int64_t n, const float* posm, const float* sph4, double* rho) {
    int64_t i;
#pragma omp parallel for schedule(static)
    for (i = 0; i < n; ++i) {
        double hi = (double)sph4[4 * i + 0];
        double sum = 0.0;
        for (int64_t k = 0; k < n; ++k) sum += (double)posm[4 * k + 3] * sph_w(dist(posm, i, k), hi);
        rho[i] = sum;
    }
}

static void hydro_term(const float* posm, const float* sph4, int64_t i, int64_t k, double* a, double* scale) {
    if (k == i) return;
    double r = dist(posm, i, k);
    if (!(r > 0.0)) return; /* coincident pair: dW/dr(0) = 0, no direction */
    double hi = (double)sph4[4 * i + 0], hk = (double)sph4[4 * k + 0];
    double pi_ = (double)sph4[4 * i + 3], pk = (double)sph4[4 * k + 3];
    double f = -(double)posm[4 * k + 3] * (pi_ + pk) * 0.5 * (sph_dwdr(r, hi) + sph_dwdr(r, hk));
    double mag = 0.0;
    for (int d = 0; d < 3; ++d) {
        double e = ((double)posm[4 * i + d] - (double)posm[4 * k + d]) / r;
        a[d] += f * e;
        mag += (f * e) * (f * e);
    }
    *scale += sqrt(mag);
}

/* acc: 3 doubles per particle, scale: 1 per particle; only the selected groups' particles are written.
 * The rho / P/rho^2 fields of sph4 are INPUTS here (as the density pass or the caller left them). */
void orc_sph_hydro(int64_t n_sel, const int64_t* sel, const int32_t* grp_first, const int32_t* grp_n,
                   const int64_t* epj_off, const int32_t* epj_id, const float* posm, const float* sph4,
                   double* acc, double* scale) {
    int64_t s;
#pragma omp parallel for schedule(dynamic, 1)
    for (s = 0; s < n_sel; ++s) {
        int64_t g = sel ? sel[s] : s;
        int64_t first = grp_first[g], cnt = grp_n[g];
        for (int64_t i = first; i < first + cnt; ++i) {
            double a[3] = {0.0, 0.0, 0.0}, sc = 0.0;
            for (int64_t e = epj_off[g]; e < epj_off[g + 1]; ++e) hydro_term(posm, sph4, i, epj_id[e], a, &sc);
            acc[3 * i + 0] = a[0];
            acc[3 * i + 1] = a[1];
            acc[3 * i + 2] = a[2];
            scale[i] = sc;
        }
    }
}

void orc_sph_hydro_direct(int64_t n, const float* posm, const float* sph4, double* acc, double* scale) {
    int64_t i;
#pragma omp parallel for schedule(static)
    for (i = 0; i < n; ++i) {
        double a[3] = {0.0, 0.0, 0.0}, sc = 0.0;
        for (int64_t k = 0; k < n; ++k) hydro_term(posm, sph4, i, k, a, &sc);
        acc[3 * i + 0] = a[0];
        acc[3 * i + 1] = a[1];
        acc[3 * i + 2] = a[2];
        scale[i] = sc;
    }
}
