/* nb_oracle.c -- TEST INFRASTRUCTURE, not the product.
 *
 * Plain fp64 CPU statement of what the hot path computes: the Hermite predictor on the
 * j-particles ("optional prediction step on the j particles"; "4th order
 * Hermite predictor-corrector") and the direct summation of the forces that the j-particles exert
 * on the i-particles (section III.A: "the forces exerted by the j-particles onto the
 * i-particles have to be computed", cost N_i N_j).  The paper prints neither formula; the readings
 * R1..R9 taken here are listed in DESIGN.md section 3.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * call this.  It shares no code with paper_1409_5474_b200/csrc: own loops, own layout handling.
 * One double loop, j in index order, OpenMP over i only, 1/sqrt correctly rounded, no FMA
 * contraction (-ffp-contract=off), no fast-math, no tiling.
 *
 * Pins (tests/test_oracle_pins.py): exact two-body rationals (P1), momentum sums (P2), Plummer
 * W -> -1/2 (P3), finite-difference jerk (P4), acc = -grad pot (P5), 50-digit brute force at
 * N <= 64 (P6), invariances (P7), ring closed form (P8), predictor exact values and order (P9).
 * Parity unpinned: nothing.
 *
 * Layout: every vector quantity is SoA [3][n] (component-major), doubles; i_list is int32.
 */
#include <math.h>
#include <stdint.h>

/* R1: Taylor series from (x, v, a, jerk) stored at t_j to time t.
 *   xp = x + v dt + a dt^2/2 + jerk dt^3/6 ,  vp = v + a dt + jerk dt^2/2 ,  dt = t - t_j. */
void oracle_predict(int64_t n, double t, const double *x, const double *v, const double *a,
                    const double *jk, const double *tj, double *xp, double *vp)
{
    #pragma omp parallel for schedule(static)
    for (int64_t p = 0; p < n; ++p) {
        double dt = t - tj[p];
        double dt2h = dt * dt / 2.0;
        double dt3s = dt * dt * dt / 6.0;
        for (int c = 0; c < 3; ++c) {
            int64_t q = (int64_t)c * n + p;
            xp[q] = x[q] + v[q] * dt + a[q] * dt2h + jk[q] * dt3s;
            vp[q] = v[q] + a[q] * dt + jk[q] * dt2h;
        }
    }
}

/* R2 (Newtonian gravity, Plummer softening, G = 1), R4 (pot excludes self), R5 (self excluded by
 * index identity), R6 (s == 0 contributes nothing), R7 (pair unsoftened iff both flagged).
 * For each k < ni, i = ilist[k], summing j = 0..n-1 in index order, j != i:
 *   r = xp_j - xp_i, w = vp_j - vp_i, s = r.r + e2, rinv = 1/sqrt(s)
 *   pot -= m_j rinv ; acc += m_j rinv^3 r ; jrk += m_j rinv^3 ( w - 3 (r.w) rinv^2 r ). */
void oracle_force(int64_t n, const double *m, const double *xp, const double *vp,
                  const uint8_t *flags, int64_t ni, const int32_t *ilist, double eps2,
                  double *acc, double *jrk, double *pot)
{
    const double *X = xp, *Y = xp + n, *Z = xp + 2 * n;
    const double *U = vp, *V = vp + n, *W = vp + 2 * n;
    #pragma omp parallel for schedule(dynamic, 16)
    for (int64_t k = 0; k < ni; ++k) {
        int64_t i = ilist[k];
        double xi = X[i], yi = Y[i], zi = Z[i], ui = U[i], vi = V[i], wi = W[i];
        int fi = flags ? (flags[i] & 1) : 0;
        double ax = 0, ay = 0, az = 0, jx = 0, jy = 0, jz = 0, p = 0;
        for (int64_t j = 0; j < n; ++j) {
            if (j == i) continue;
            double rx = X[j] - xi, ry = Y[j] - yi, rz = Z[j] - zi;
            double wx = U[j] - ui, wy = V[j] - vi, wz = W[j] - wi;
            double e2 = (fi && (flags[j] & 1)) ? 0.0 : eps2;
            double s = rx * rx + ry * ry + rz * rz + e2;
            if (s == 0.0) continue;
            double rinv = 1.0 / sqrt(s);
            double rinv2 = rinv * rinv;
            double mr = m[j] * rinv;
            double mr3 = mr * rinv2;
            double b = 3.0 * (rx * wx + ry * wy + rz * wz) * rinv2;
            p -= mr;
            ax += mr3 * rx;
            ay += mr3 * ry;
            az += mr3 * rz;
            jx += mr3 * (wx - b * rx);
            jy += mr3 * (wy - b * ry);
            jz += mr3 * (wz - b * rz);
        }
        acc[k] = ax; acc[ni + k] = ay; acc[2 * ni + k] = az;
        jrk[k] = jx; jrk[ni + k] = jy; jrk[2 * ni + k] = jz;
        pot[k] = p;
    }
}

/* How many OpenMP threads the two functions above will use (for the cpu_baseline report). */
#ifdef _OPENMP
#include <omp.h>
int oracle_threads(void) { return omp_get_max_threads(); }
#else
int oracle_threads(void) { return 1; }
#endif
