/*
 * CPU ORACLE for the O(N) neighbours of the kick in GENGA's hybrid symplectic step
 * (Rcrit, HC, FG).            *** TEST INFRASTRUCTURE ONLY ***
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * call this file.  It shares no code, header, table or helper with the CUDA path in
 * paper_2201_10058_b200/csrc/ and neither includes the other.
 *
 * What it computes (each is the plain definition, evaluated in long double and rounded once):
 *
 *   Rcrit  r_crit,i^(k) = max(n1 R_H,i , n2 (dt / s^k) v_i),  k = 0..nrows-1      eq. 5 PAPER.md:72-76;
 *          "the critical radius is defined in the same way on each level ... with the reduced
 *          time step" PAPER.md:638.  R_H,i = a_i (m_i / (3 m_star))^(1/3) with a_i the osculating
 *          semi-major axis from the vis-viva equation, v_i = |v_i|               (reading G6)
 *   HC     q_i += dt * (sum_j m_j v_j) / m_star            eq. 4 PAPER.md:68 (H_C = (sum p)^2 / 2 m_star,
 *          dq_i/dt = dH_C/dp_i), "the democratic momentum summation" App. A
 *   FG     every body advances by dt on its two-body orbit about the central mass with
 *          mu = G m_star (the Kepler part p^2/2m - G m m_star / r of eq. 2; the
 *          pair term [1 - K] of eq. 2 belongs to the Bulirsch-Stoer phase, off this path).
 *          The exact solution is written with Gauss' f and g functions in the difference dE of
 *          the eccentric anomaly ("FG", App. A); a body on a hyperbolic orbit
 *          (1/a < 0: ejected, or above the escape speed inside a deep passage) follows the same
 *          two-body solution in the difference dH of the hyperbolic anomaly; only the parabolic
 *          case 1/a = 0 exactly is left untouched and reported                    (reading G13)
 *   step   Rcrit(dt); Kick(dt/2) + pre-check; HC(dt/2); FG(dt); HC(dt/2); Kick(dt/2)
 *          App. A PAPER.md:986-992 without the Bulirsch-Stoer branch -- composed in Python
 *          (oracle/step.py) from these functions and genga_oracle_kick.
 *
 * PINS (tests/test_step_oracle_pins.py, `-m "not gpu"`): n1 = 3, n2 = 0.4 and the closed form of
 * eq. 5 on a circular orbit; HC on a hand-computed 3-body example and conservation of sum p; FG
 * against the closed-form rotation of a circular orbit, against the input generator's
 * elements -> Cartesian map at M0 + n dt (an independent Kepler solver), conservation of energy,
 * angular momentum and eccentricity vector, a full period, and dt followed by -dt; the whole step:
 * dt^2 scaling of the energy error of a 3-body system (P8 with the oracle's own HC and FG).
 */
#include <math.h>
#include <stdint.h>

/* eq. 5, rows k = 0..nrows-1 at dt / substeps^k.  out [nrows][N].  Returns the number of bodies
 * with a non-positive semi-major axis (their Hill term is taken as 0). */
int64_t genga_oracle_rcrit(int64_t N, const double *pos, const double *vel, const double *mass,
                           double m_star, double G, double dt, double substeps, int32_t nrows,
                           double n1, double n2, double *out)
{
    int64_t unbound = 0;
    for (int64_t i = 0; i < N; i++) {
        const long double x = pos[i], y = pos[N + i], z = pos[2 * N + i];
        const long double vx = vel[i], vy = vel[N + i], vz = vel[2 * N + i];
        const long double r = sqrtl(x * x + y * y + z * z);
        const long double v2 = vx * vx + vy * vy + vz * vz;
        const long double mu = (long double)G * (long double)m_star;
        const long double inv_a = 2.0L / r - v2 / mu;                  /* vis-viva */
        long double hill = 0.0L;
        if (inv_a > 0.0L) hill = (1.0L / inv_a) * cbrtl((long double)mass[i] / (3.0L * (long double)m_star));
        else unbound++;
        const long double v = sqrtl(v2);
        long double dtk = dt;
        for (int32_t k = 0; k < nrows; k++) {
            const long double a = (long double)n1 * hill, b = (long double)n2 * dtk * v;
            out[(int64_t)k * N + i] = (double)(a > b ? a : b);
            dtk /= (long double)substeps;
        }
    }
    return unbound;
}

/* eq. 4: q_i += dt * (sum_j m_j v_j) / m_star.  psum (if not NULL) receives sum_j m_j v_j. */
void genga_oracle_hc(int64_t N, double *pos, const double *vel, const double *mass, double m_star,
                     double dt, double *psum)
{
    long double p[3] = {0.0L, 0.0L, 0.0L};
    for (int c = 0; c < 3; c++)
        for (int64_t j = 0; j < N; j++) p[c] += (long double)mass[j] * (long double)vel[c * N + j];
    for (int c = 0; c < 3; c++) {
        const long double shift = (long double)dt * p[c] / (long double)m_star;
        for (int64_t i = 0; i < N; i++) pos[c * N + i] = (double)((long double)pos[c * N + i] + shift);
        if (psum) psum[c] = (double)p[c];
    }
}

/* The Kepler drift of one body, long double.  Returns 0, or 1 if the orbit is parabolic (left untouched). */
static int kepler_step(long double mu, long double dt, long double q[3], long double v[3])
{
    const long double r0 = sqrtl(q[0] * q[0] + q[1] * q[1] + q[2] * q[2]);
    const long double v2 = v[0] * v[0] + v[1] * v[1] + v[2] * v[2];
    const long double u = q[0] * v[0] + q[1] * v[1] + q[2] * v[2];
    const long double inv_a = 2.0L / r0 - v2 / mu;
    if (inv_a < 0.0L) {
        /* hyperbolic: a' = -a > 0, n' = sqrt(mu / a'^3); Kepler's equation in the difference dH = H - H0:
         *   F(dH) = ec sinh dH + es (cosh dH - 1) - dH - n' dt = 0,   ec = e cosh H0 = 1 + r0/a',  es = e sinh H0 = u / (n' a'^2)
         * F' = ec cosh dH + es sinh dH - 1 = r/a' > 0: increasing.  Bracket by doubling, bisection, two Newton steps.
         *   r = a' (ec cosh dH + es sinh dH - 1),  f = 1 - (a'/r0)(cosh dH - 1),  g = dt - (sinh dH - dH)/n',
         *   f' = -(a'^2 n' / (r0 r)) sinh dH,      g' = 1 - (a'/r)(cosh dH - 1) */
        const long double ap = -1.0L / inv_a;
        const long double np_ = sqrtl(mu / (ap * ap * ap));
        const long double ec = 1.0L + r0 / ap, es = u / (np_ * ap * ap), dN = np_ * dt;
        long double lo = 0.0L, hi = 0.0L, w = 1.0L;
        for (int it = 0; it < 64; it++) {
            const long double x = dN > 0.0L ? w : -w;
            const long double fn = ec * sinhl(x) + es * (coshl(x) - 1.0L) - x - dN;
            if (dN > 0.0L ? fn >= 0.0L : fn <= 0.0L) { if (dN > 0.0L) hi = x; else lo = x; break; }
            if (dN > 0.0L) lo = x; else hi = x;
            w *= 2.0L;
        }
        long double dH = 0.5L * (lo + hi);
        for (int it = 0; it < 200; it++) {
            dH = 0.5L * (lo + hi);
            if (!(dH > lo && dH < hi)) break;
            const long double fn = ec * sinhl(dH) + es * (coshl(dH) - 1.0L) - dH - dN;
            if (fn > 0.0L) hi = dH; else lo = dH;
        }
        for (int it = 0; it < 2; it++) {
            const long double sh = sinhl(dH), ch = coshl(dH);
            const long double nx = dH - (ec * sh + es * (ch - 1.0L) - dH - dN) / (ec * ch + es * sh - 1.0L);
            if (nx >= lo && nx <= hi) dH = nx;
        }
        const long double sh = sinhl(dH), ch = coshl(dH);
        const long double r = ap * (ec * ch + es * sh - 1.0L);
        const long double f = 1.0L - (ap / r0) * (ch - 1.0L);
        const long double g = dt - (sh - dH) / np_;
        const long double fd = -(ap * ap * np_ / (r0 * r)) * sh;
        const long double gd = 1.0L - (ap / r) * (ch - 1.0L);
        for (int k = 0; k < 3; k++) {
            const long double qk = f * q[k] + g * v[k];
            const long double vk = fd * q[k] + gd * v[k];
            q[k] = qk;
            v[k] = vk;
        }
        return 0;
    }
    if (!(inv_a > 0.0L)) return 1;                                     /* parabolic (or not a number) */
    const long double a = 1.0L / inv_a;
    const long double n = sqrtl(mu / (a * a * a));                     /* mean motion */
    const long double ec = 1.0L - r0 / a;                              /* e cos E0 */
    const long double es = u / (n * a * a);                            /* e sin E0 */
    const long double dM = n * dt;
    /* Kepler's equation in the difference dE = E - E0:
     *   F(dE) = dE - ec sin dE + es (1 - cos dE) - dM = 0.
     * F' = 1 - ec cos dE + es sin dE = r/a > 0, so F is increasing, and |F(dE) - (dE - dM)| <= |ec| + 2|es|:
     * the root is bracketed by dM -+ (|ec| + 2|es|).  Plain bisection to the last bit of the bracket
     * (slow, cannot fail), then two Newton steps to polish. */
    long double lo = dM - (fabsl(ec) + 2.0L * fabsl(es)) - 1e-300L, hi = dM + (fabsl(ec) + 2.0L * fabsl(es)) + 1e-300L;
    long double dE = 0.5L * (lo + hi);
    for (int it = 0; it < 200; it++) {
        dE = 0.5L * (lo + hi);
        if (!(dE > lo && dE < hi)) break;
        const long double fn = (dE - dM) - ec * sinl(dE) + es * (1.0L - cosl(dE));
        if (fn > 0.0L) hi = dE; else lo = dE;
    }
    for (int it = 0; it < 2; it++) {
        const long double s = sinl(dE), c = cosl(dE);
        const long double fn = (dE - dM) - ec * s + es * (1.0L - c);
        const long double fp = 1.0L - ec * c + es * s;
        const long double nx = dE - fn / fp;
        if (nx >= lo && nx <= hi) dE = nx;
    }
    const long double s = sinl(dE), c = cosl(dE);
    const long double r = a * (1.0L - ec * c + es * s);
    const long double f = 1.0L - (a / r0) * (1.0L - c);
    const long double g = dt + (s - dE) / n;
    const long double fd = -(a * a * n / (r0 * r)) * s;
    const long double gd = 1.0L - (a / r) * (1.0L - c);
    for (int k = 0; k < 3; k++) {
        const long double qk = f * q[k] + g * v[k];
        const long double vk = fd * q[k] + gd * v[k];
        q[k] = qk;
        v[k] = vk;
    }
    return 0;
}

/* FG(dt) for all bodies, in place.  Returns the number of bodies on a parabolic orbit (1/a = 0
 * exactly: left untouched). */
int64_t genga_oracle_fg(int64_t N, double *pos, double *vel, double mu, double dt)
{
    int64_t unbound = 0;
#pragma omp parallel for schedule(static) reduction(+ : unbound)
    for (int64_t i = 0; i < N; i++) {
        long double q[3] = {pos[i], pos[N + i], pos[2 * N + i]};
        long double v[3] = {vel[i], vel[N + i], vel[2 * N + i]};
        if (kepler_step((long double)mu, (long double)dt, q, v)) { unbound++; continue; }
        for (int k = 0; k < 3; k++) {
            pos[k * N + i] = (double)q[k];
            vel[k * N + i] = (double)v[k];
        }
    }
    return unbound;
}
