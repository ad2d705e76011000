/*
 * CPU ORACLE for the close-encounter detection after the Kepler drift (SURVEY.md 8(f) NEXT-2,
 * first half).                                         *** TEST INFRASTRUCTURE ONLY ***
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * call this file.  It shares no code, header, table or helper with the CUDA path in
 * paper_2201_10058_b200/csrc/ and neither includes the other.
 *
 * App. A: "FG(dt); if (close-encounter candidates): close-encounter detection;
 * if (close-encounters): grouping; Bulirsch-Stoer(dt)".  The pre-check fused in the kick over-selects
 * candidates from the positions BEFORE the drift; the detection decides, with the states before and
 * after the drift in hand, which candidates are close-encounter pairs of this step.
 *
 * PARITY UNPINNED (reading G16): PAPER.md names the step and prints no criterion (it refers
 * to Grimm & Stadel 2014).  The reading taken is the one of the hybrid integrator the paper builds on
 * (Chambers 1999, the paper's reference for K and r_crit): a candidate {i, j} is a close-encounter pair
 * if the MINIMUM over the step of the cubic Hermite interpolant of the squared separation lies inside
 * the pair's critical radius,
 *
 *     p(tau), tau in [0, 1]:  p(0) = d0 = |q_j - q_i|^2 before the drift,  p(1) = d1 after it,
 *                             p'(0) = m0 = h * 2 (q_j - q_i).(v_j - v_i) before,  p'(1) = m1 after
 *     p(tau) = a tau^3 + b tau^2 + c tau + d0,   a = 2 d0 - 2 d1 + m0 + m1,
 *                                                b = 3 d1 - 3 d0 - 2 m0 - m1,   c = m0
 *     encounter  <=>  min(d0, d1, p(tau*) if 0 < tau* < 1) < (f * max(rc_i, rc_j))^2
 *
 * where tau* is the root of p'(tau) = 3 a tau^2 + 2 b tau + c with p'' >= 0 (the local minimum):
 * tau* = (-b + sqrt(b^2 - 3 a c)) / (3 a), written as -c / (b + sqrt(..)) when b > 0 (the same root;
 * no cancellation when a -> 0, i.e. for nearly uniform relative motion, where p is a parabola).
 * What the mathematics fixes is pinned (tests/test_detect_oracle_pins.py): the interpolation
 * conditions, the exact closest approach for uniform relative motion, the minimum against a dense
 * scan of scipy's CubicHermiteSpline, symmetry under i <-> j and under time reversal, counts.
 * The CHOICE of this criterion is what the paper does not pin.
 *
 * All arithmetic is IEEE binary64, one rounding per operation, in the order written (the decision
 * is an integer taken from floating point: the CUDA path takes it in the same precision and order).
 */
#include <math.h>
#include <stdint.h>

/* min over [0, 1] of the cubic Hermite interpolant through (d0, m0) at 0 and (d1, m1) at 1 */
double genga_oracle_hermite_min(double d0, double m0, double d1, double m1, double *tau_out)
{
    double a = ((2.0 * d0 - 2.0 * d1) + m0) + m1;
    double b = ((3.0 * d1 - 3.0 * d0) - 2.0 * m0) - m1;
    double c = m0;
    double dmin = d0 <= d1 ? d0 : d1;
    double tmin = d0 <= d1 ? 0.0 : 1.0;
    double disc = b * b - (3.0 * a) * c;
    if (disc >= 0.0) {
        double s = sqrt(disc), tau = -1.0;
        if (b > 0.0) tau = -c / (b + s);
        else if (a != 0.0) tau = (s - b) / (3.0 * a);
        if (tau > 0.0 && tau < 1.0) {
            double p = ((a * tau + b) * tau + c) * tau + d0;
            if (p < dmin) { dmin = p; tmin = tau; }
        }
    }
    if (tau_out) *tau_out = tmin;
    return dmin;
}

/*
 * pos0, vel0: [3][N] before the drift; pos1, vel1: after it; rc_row [N]; h = the drift's dt.
 * pairs [npairs][2].  Outputs: enc [npairs] (1 = close-encounter pair), border [npairs]
 * (|sqrt(dmin) / (f rc) - 1| <= 1e-12), d2min [npairs], count [N] (encounter pairs per body).
 * Returns the number of encounter pairs.
 */
int64_t genga_oracle_detect(int64_t N, const double *pos0, const double *vel0, const double *pos1,
                            const double *vel1, const double *rc_row, double enc_factor, double h,
                            const int32_t *pairs, int64_t npairs, int8_t *enc, int8_t *border,
                            double *d2min, int32_t *count)
{
    int64_t total = 0;
    for (int64_t i = 0; i < N; i++) count[i] = 0;
    for (int64_t q = 0; q < npairs; q++) {
        int64_t i = pairs[2 * q], j = pairs[2 * q + 1];
        double d[2], m[2];
        for (int s = 0; s < 2; s++) {
            const double *P = s ? pos1 : pos0, *V = s ? vel1 : vel0;
            double dx = P[j] - P[i], dy = P[N + j] - P[N + i], dz = P[2 * N + j] - P[2 * N + i];
            double ux = V[j] - V[i], uy = V[N + j] - V[N + i], uz = V[2 * N + j] - V[2 * N + i];
            d[s] = dx * dx + dy * dy + dz * dz;
            m[s] = h * (2.0 * (dx * ux + dy * uy + dz * uz));
        }
        double dm = genga_oracle_hermite_min(d[0], m[0], d[1], m[1], 0);
        double rc = rc_row[i] >= rc_row[j] ? rc_row[i] : rc_row[j];
        double R = enc_factor * rc;
        int e = dm < R * R;
        enc[q] = (int8_t)e;
        border[q] = (int8_t)(dm > 0.0 && fabs(sqrt(dm) / R - 1.0) <= 1e-12);
        d2min[q] = dm;
        if (e) { count[i]++; count[j]++; total++; }
    }
    return total;
}
