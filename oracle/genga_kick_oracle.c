/*
 * CPU ORACLE for the GENGA kick + close-encounter pre-check.   *** TEST INFRASTRUCTURE ONLY ***
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * call this file.  It shares no code, header, table or helper with the CUDA path in
 * paper_2201_10058_b200/csrc/ and neither includes the other.
 *
 * What it computes is the PLAIN DEFINITION of the path (the method is an exact direct sum, so
 * the oracle is that sum written out):
 *
 *   a_i = sum_{j in J(i), j != i}  G m_j W(r_ij) (x_j - x_i) / r_ij^3        eq. 3
 *                                                                            (force-weighted, reading G5)
 *   W   = prod_{k<L} [1 - K(r; rc_k)] * K(r; rc_L)                           eq. 62-63
 *                                                                            (telescoping product, reading G3)
 *   K(r; rc): y = (r - 0.1 rc)/(0.9 rc); 0 if y<=0; 1 if y>=1;
 *             else y^2/(2y^2 - 2y + 1)
 *                                                                            (form of Chambers 1999 eq. 10,
 *                                                                             NOT printed in PAPER.md: reading G1)
 *   rc_k for a pair = max(rcrit[k][i], rcrit[k][j])                          reading G2 (parity unpinned)
 *   pre-check: partner iff r2 < (f * rc_L)^2, strict                         App. A, reading G4
 *                                                                            (f: parity unpinned)
 *   J(i) = massive bodies [0, n_massive) for every i (semi-active test
 *   particles feel the massive bodies, not each other)                       sec. 8.1
 *   A massive body also lists its test-particle partners (reading G11).  tp_mode selects the force
 *   terms of Fig. 14: 1 = "TP 1", test particles exert no force (the rectangular
 *   kick of north_star, reading G10); 2 = "TP 2", semi-active particles with mass also act on the
 *   massive bodies "the same way as in the fully interactive mode": massive i
 *   then sums over ALL j.
 *
 * Arithmetic: every per-pair quantity in IEEE binary64 exactly in the order written below
 * (compile with -ffp-contract=off); the sums over j in long double (x87 80-bit, 64-bit
 * significand), rounded to binary64 once at the end.
 *
 * PINS (tests/test_oracle_pins.py, all `-m "not gpu"`): two-body closed form (P1), exact rational
 * values / symmetry / C1-continuity of K (P2), momentum (P3), Newtonian limit vs an independently
 * written numpy sum (P4), partition of unity of the level weights (P5), "<= 2 levels active" for
 * s = 10 (P6), level-1 closed form max 1/4 (P7), dt^2 energy scaling of a 3-body leapfrog (P8),
 * the Fig. 7 ring with exactly 8 partners (P9), 50-digit mpmath brute force on N <= 8 (P10).
 * Unpinned by the paper (stated in DESIGN.md): the choice max() in G2 and the factor f in G4.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* Changeover function K as a function of y = (r - 0.1 rc)/(0.9 rc).   reading G1 */
double genga_oracle_K_of_y(double y)
{
    if (y <= 0.0) return 0.0;
    if (y >= 1.0) return 1.0;
    return (y * y) / (2.0 * y * y - 2.0 * y + 1.0);
}

/* K(r; rc)   PAPER.md:70, :619 ("acting in the range 0.1 < r/rcrit < 1.0"), :642 */
double genga_oracle_K(double r, double rc)
{
    double y = (r - 0.1 * rc) / (0.9 * rc);
    return genga_oracle_K_of_y(y);
}

/* Level weight W_L for one pair; rc[k], k = 0..L, are the PAIR radii.   eq. 62-63, reading G3.
 * L = -1 is not a level; use genga_oracle_weight_bs for the Bulirsch-Stoer remainder. */
double genga_oracle_weight(double r, const double *rc, int L)
{
    double W = 1.0;
    for (int k = 0; k < L; k++) W *= (1.0 - genga_oracle_K(r, rc[k]));
    W *= genga_oracle_K(r, rc[L]);
    return W;
}

/* K_Bulirsch-Stoer for `nlevels` symplectic levels: prod_{k<nlevels} (1 - K_k).   eq. 62-63 */
double genga_oracle_weight_bs(double r, const double *rc, int nlevels)
{
    double W = 1.0;
    for (int k = 0; k < nlevels; k++) W *= (1.0 - genga_oracle_K(r, rc[k]));
    return W;
}

int genga_oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/*
 * The kick + pre-check for the bodies listed in rows[0..nrows).
 *
 *   pos   [3][N]  SoA heliocentric positions          mass [N]
 *   rcrit [L+1][N] row k = r_crit_i at dt / s^k       N = n_massive + n_test
 *   rows  [nrows] body indices to evaluate (any subset, any order)
 * outputs, all indexed by position in `rows`:
 *   acc  [3][nrows]   acceleration                    (NULL allowed)
 *   S    [3][nrows]   sum_j |term|, component-wise: the tolerance scale of north_star
 *   count[nrows]      number of encounter partners (true count, even if > maxp)
 *   partners [nrows][maxp]  partner indices j, ascending in j (first maxp of them)
 *   border   [bcap][2], *nborder: pairs (i, j) with | r/(f rc_L) - 1 | <= 1e-12 ("borderline", G4)
 * returns 0, or -1 on a coincident distinct pair (r2 == 0: outside the domain, G7).
 */
int genga_oracle_kick_tp(int32_t n_massive, int32_t n_test, int32_t tp_mode, int32_t L, double G, double f,
                      const double *pos, const double *mass, const double *rcrit,
                      const int32_t *rows, int64_t nrows,
                      double *acc, double *S, int32_t *count,
                      int32_t *partners, int32_t maxp,
                      int32_t *border, int64_t bcap, int64_t *nborder)
{
    const int64_t N = (int64_t)n_massive + (int64_t)n_test;
    const double *x = pos, *y = pos + N, *z = pos + 2 * N;
    int bad = 0;
    int64_t nb = 0;

#pragma omp parallel for schedule(static)
    for (int64_t q = 0; q < nrows; q++) {
        const int64_t i = rows[q];
        const int i_massive = i < n_massive;
        long double ax = 0.0L, ay = 0.0L, az = 0.0L, sx = 0.0L, sy = 0.0L, sz = 0.0L;
        int32_t cnt = 0;
        /* massive i: force from massive j, encounter check against ALL bodies;
         * test i   : force from and encounter check against massive j only.     sec. 8.1 */
        const int64_t jend = i_massive ? N : n_massive;
        for (int64_t j = 0; j < jend; j++) {
            if (j == i) continue;                                   /* G7: skip by index */
            const double dx = x[j] - x[i];
            const double dy = y[j] - y[i];
            const double dz = z[j] - z[i];
            const double r2 = dx * dx + dy * dy + dz * dz;
            if (!(r2 > 0.0)) { bad = 1; continue; }
            const double r = sqrt(r2);
            /* pre-check on the level-L pair radius   (G2, G4) */
            const double rcL = fmax(rcrit[(int64_t)L * N + i], rcrit[(int64_t)L * N + j]);
            const double thr = f * rcL;
            if (r2 < thr * thr) {
                if (cnt < maxp && partners) partners[q * (int64_t)maxp + cnt] = (int32_t)j;
                cnt++;
            }
            if (border && fabs(r / thr - 1.0) <= 1e-12) {
                int64_t slot;
#pragma omp atomic capture
                slot = nb++;
                if (slot < bcap) { border[2 * slot] = (int32_t)i; border[2 * slot + 1] = (int32_t)j; }
            }
            if (j >= n_massive && tp_mode != 2) continue;           /* TP 1: no force from test particles */
            /* level weight   (eq. 62-63, G3) */
            double W = 1.0;
            for (int k = 0; k < L; k++) {
                const double rck = fmax(rcrit[(int64_t)k * N + i], rcrit[(int64_t)k * N + j]);
                W *= (1.0 - genga_oracle_K(r, rck));
            }
            W *= genga_oracle_K(r, rcL);
            if (W == 0.0) continue;                                 /* G7: no 0 * inf */
            const double s = G * mass[j] * W / (r2 * r);            /* eq. 3, G5, G8 */
            const double tx = s * dx, ty = s * dy, tz = s * dz;
            ax += tx; ay += ty; az += tz;
            sx += fabs(tx); sy += fabs(ty); sz += fabs(tz);
        }
        if (acc) { acc[q] = (double)ax; acc[nrows + q] = (double)ay; acc[2 * nrows + q] = (double)az; }
        if (S)   { S[q] = (double)sx;   S[nrows + q] = (double)sy;   S[2 * nrows + q] = (double)sz; }
        if (count) count[q] = cnt;
    }
    if (nborder) *nborder = nb;
    return bad ? -1 : 0;
}

/* TP 1 (the rectangular kick of north_star): the entry point the kick tests use. */
int genga_oracle_kick(int32_t n_massive, int32_t n_test, int32_t L, double G, double f,
                      const double *pos, const double *mass, const double *rcrit,
                      const int32_t *rows, int64_t nrows,
                      double *acc, double *S, int32_t *count,
                      int32_t *partners, int32_t maxp,
                      int32_t *border, int64_t bcap, int64_t *nborder)
{
    return genga_oracle_kick_tp(n_massive, n_test, 1, L, G, f, pos, mass, rcrit, rows, nrows, acc, S, count,
                                partners, maxp, border, bcap, nborder);
}

/*
 * KickS (App. A: "KickS ... similar to the original functions, but applied only to
 * the relevant bodies in each symplectic level"; groupS "extracts all relevant close-encounter pairs
 * from the upper symplectic level"): the sum of eq. 3 with the level weight W_L of eq. 62-63 over the
 * pairs of a LIST (each unordered pair once, rows (i, j), i != j) instead of over all pairs, both
 * directions of each pair, and the level-L pre-check of the listed pairs.
 * Per-pair arithmetic exactly as in genga_oracle_kick_tp, from each body's own side (d = x_other - x_self).
 * Force rules (sec. 8.1): a test particle feels massive bodies only; it acts on a massive body only
 * if tp_mode == 2; two test particles do not interact.
 *   acc, S [3][N] (all bodies; bodies in no pair get 0), count [N], enc [n_pairs] (1 if the pair is a
 *   level-L encounter pair), border [n_pairs] (1 if within 1e-12 of the threshold).
 * Since W_L = 0 for r >= rc0_ij (factor 1 - K_0), this equals the all-pairs level-L kick (L >= 1)
 * whenever the list holds every pair with r < rc0_ij -- the pin of tests/test_oracle_pins.py.
 * returns 0, or -1 on a coincident pair.
 */
int genga_oracle_kick_list(int32_t n_massive, int32_t n_test, int32_t tp_mode, int32_t L, double G, double f,
                           const double *pos, const double *mass, const double *rcrit,
                           const int32_t *pairs, int64_t n_pairs,
                           double *acc, double *S, int32_t *count, int8_t *enc, int8_t *border)
{
    const int64_t N = (int64_t)n_massive + (int64_t)n_test;
    const double *x = pos, *y = pos + N, *z = pos + 2 * N;
    long double *a = (long double *)calloc((size_t)(6 * N > 0 ? 6 * N : 1), sizeof(long double));
    long double *s_abs = a + 3 * N;
    int bad = 0;
    for (int64_t i = 0; i < N; i++) count[i] = 0;
    for (int64_t p = 0; p < n_pairs; p++) {
        enc[p] = 0; border[p] = 0;
        for (int side = 0; side < 2; side++) {
            const int64_t i = pairs[2 * p + side], j = pairs[2 * p + 1 - side];      /* i feels j */
            if (i == j) continue;
            const double dx = x[j] - x[i];
            const double dy = y[j] - y[i];
            const double dz = z[j] - z[i];
            const double r2 = dx * dx + dy * dy + dz * dz;
            if (!(r2 > 0.0)) { bad = 1; continue; }
            const double r = sqrt(r2);
            const double rcL = fmax(rcrit[(int64_t)L * N + i], rcrit[(int64_t)L * N + j]);
            const double thr = f * rcL;
            const int both_tp = i >= n_massive && j >= n_massive;
            if (r2 < thr * thr && !both_tp) { count[i]++; enc[p] = 1; }
            if (fabs(r / thr - 1.0) <= 1e-12) border[p] = 1;
            if (both_tp) continue;
            if (j >= n_massive && tp_mode != 2) continue;             /* no force from a test particle (TP 1) */
            double W = 1.0;
            for (int k = 0; k < L; k++) {
                const double rck = fmax(rcrit[(int64_t)k * N + i], rcrit[(int64_t)k * N + j]);
                W *= (1.0 - genga_oracle_K(r, rck));
            }
            W *= genga_oracle_K(r, rcL);
            if (W == 0.0) continue;
            const double s = G * mass[j] * W / (r2 * r);
            const double tx = s * dx, ty = s * dy, tz = s * dz;
            a[i] += tx; a[N + i] += ty; a[2 * N + i] += tz;
            s_abs[i] += fabs(tx); s_abs[N + i] += fabs(ty); s_abs[2 * N + i] += fabs(tz);
        }
    }
    for (int64_t q = 0; q < 3 * N; q++) { acc[q] = (double)a[q]; S[q] = (double)s_abs[q]; }
    free(a);
    return bad ? -1 : 0;
}
