/*
 * CPU ORACLE for the Bulirsch-Stoer integration of close-encounter groups (SURVEY.md 8(f) NEXT-4,
 * last item; "we also use a Bulirsch-Stoer ... method to resolve the close-encounter
 * part", :559 "All particles in a given close-encounter group need to be integrated synchronously",
 * App. A PAPER.md:989 "Bulirsch-Stoer(dt)").            *** TEST INFRASTRUCTURE ONLY ***
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call
 * this file.  It shares no code, header, table or helper with the CUDA path.
 *
 * What is integrated.  The part H_A of the Hamiltonian (eq. 2) restricted to the
 * bodies of ONE group, over the step dt, starting from the state BEFORE the Kepler drift:
 *     dq_i/dt = v_i
 *     dv_i/dt = - G m_star q_i / |q_i|^3  +  sum_{j in group, j != i}  G m_j W_BS(r_ij) (q_j - q_i) / r_ij^3
 *     W_BS    = prod_{k < nlevels} [1 - K(r_ij; rck_ij)]      K_Bulirsch-Stoer of eq. 62-63;
 *               nlevels = 1: the complement 1 - K of the kick's weight, so that kick + this = Newton
 * (force-weighted like the kick, reading G5; rck_ij = max of the two bodies' rows, reading G2;
 * Test-particle modes, sec. 8.1 PAPER.md:791-808 and Fig. 14: with is_tp given, the term of j on i is summed iff j is a
 * massive body, or j is a semi-active particle, the mode is TP 2 and i is a massive body -- particles feel the massive
 * bodies "the same way as in the fully interactive mode", act on them only in TP 2, and never feel each other.)
 *
 * How.  PAPER.md names the method and gives no algorithmic detail (it refers to Grimm & Stadel 2014 and
 * to textbooks); the scheme below is the textbook Gragg-Bulirsch-Stoer method, fixed here as reading G15
 * (DESIGN.md):
 *   - one macro step of length H: modified midpoint rule with n_k = 2 k sub-steps, k = 1 .. 8,
 *         z_0 = y;  z_1 = z_0 + h f(z_0);  z_{m+1} = z_{m-1} + 2 h f(z_m);  y_k = (z_n + z_{n-1} + h f(z_n)) / 2,  h = H / n_k
 *   - polynomial extrapolation in h^2 (Aitken-Neville):  T_{k,0} = y_k,
 *         T_{k,j} = T_{k,j-1} + (T_{k,j-1} - T_{k-1,j-1}) / ((n_k / n_{k-j})^2 - 1)
 *   - error of column k >= 2: err = max over the group's bodies of
 *         max( |T_kk - T_k,k-1|_q / |T_kk|_q ,  |T_kk - T_k,k-1|_v / |T_kk|_v )      (Euclidean norms per body)
 *     accept T_kk as soon as err <= tol; if k = 8 is not enough, halve H and start the macro step again
 *   - after an accepted macro step: H <- 2 H if it converged with k <= 5, else H; never beyond the end of dt.
 *     The first macro step tries the whole dt.
 * All arithmetic in IEEE binary64 in the order written (compile with -ffp-contract=off).  The force on a body is
 * the plain sum of its definition: the Sun term, then the pair terms added one by one in member order
 * j = 0 .. n-1, for every group size.  The oracle knows nothing of how a kernel spreads that sum over threads: a kernel
 * that sums in another order differs from this file at rounding level, and the parity tests bound that difference
 * (tests/test_gpu_bs.py) instead of asking for equal bits.  Single-threaded.
 *
 * PINS (tests/test_bs_oracle_pins.py): two bodies far outside each other's critical radius (W_BS = 0):
 * each follows its Kepler orbit -- against the closed-form FG oracle; two bodies deep inside (K = 0): the
 * Newtonian three-body energy (Sun fixed) is conserved to the tolerance; a three-body group inside the
 * changeover band against scipy's DOP853 on an independently written right-hand side; dt followed by -dt;
 * tolerance scaling.  The algorithmic choices (sequence, error norm, step control) are readings:
 * **parity unpinned** by the paper, pinned against the ODE's solution.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>

#define BS_KMAX 8
#define BS_MAX_HALVINGS 60

extern double genga_oracle_K(double r, double rc);

typedef struct {
    int n, nlevels;
    double G, mu;
    const double *m;        /* [n] */
    const double *rc;       /* [nlevels][n] */
    const int8_t *is_tp;    /* [n] 1 = semi-active test particle, or NULL (fully interactive, TP 0) */
    int tp_mode;            /* 2: particles act on the massive bodies; otherwise on nobody */
} bs_group;

/* f: accelerations of all bodies of the group at positions q [n][3] */
static void bs_accel(const bs_group *g, const double *q, double *a)
{
    const int n = g->n;
    for (int i = 0; i < n; i++) {
        const double x = q[3 * i], y = q[3 * i + 1], z = q[3 * i + 2];
        const double r2s = x * x + y * y + z * z;
        const double rs = sqrt(r2s);
        const double s0 = -g->mu / (r2s * rs);
        double ax = s0 * x, ay = s0 * y, az = s0 * z;
        for (int j = 0; j < n; j++) {
            if (j == i) continue;
            if (g->is_tp && g->is_tp[j] && (g->tp_mode != 2 || g->is_tp[i])) continue;      /* Fig. 14 */
            const double dx = q[3 * j] - x, dy = q[3 * j + 1] - y, dz = q[3 * j + 2] - z;
            const double r2 = dx * dx + dy * dy + dz * dz;
            const double r = sqrt(r2);
            double W = 1.0;
            for (int k = 0; k < g->nlevels; k++) {
                const double rck = fmax(g->rc[k * n + i], g->rc[k * n + j]);
                W *= (1.0 - genga_oracle_K(r, rck));
            }
            if (W != 0.0) {
                const double s = g->G * g->m[j] * W / (r2 * r);
                ax = ax + s * dx; ay = ay + s * dy; az = az + s * dz;
            }
        }
        a[3 * i] = ax; a[3 * i + 1] = ay; a[3 * i + 2] = az;
    }
}

/* modified midpoint over H with nsub sub-steps: (q0, v0) -> (qo, vo) */
static void bs_midpoint(const bs_group *g, const double *q0, const double *v0, const double *a0, double H, int nsub,
                        double *qo, double *vo, double *w)
{
    const int n3 = 3 * g->n;
    double *qm = w, *vm = w + n3, *qn = w + 2 * n3, *vn = w + 3 * n3, *a = w + 4 * n3;
    const double h = H / (double)nsub, h2 = 2.0 * h;
    for (int c = 0; c < n3; c++) { qm[c] = q0[c]; vm[c] = v0[c]; qn[c] = q0[c] + h * v0[c]; vn[c] = v0[c] + h * a0[c]; }
    for (int m = 1; m < nsub; m++) {
        bs_accel(g, qn, a);
        for (int c = 0; c < n3; c++) {
            const double qs = qm[c] + h2 * vn[c], vs = vm[c] + h2 * a[c];
            qm[c] = qn[c]; vm[c] = vn[c]; qn[c] = qs; vn[c] = vs;
        }
    }
    bs_accel(g, qn, a);
    for (int c = 0; c < n3; c++) {
        qo[c] = 0.5 * (qn[c] + qm[c] + h * vn[c]);
        vo[c] = 0.5 * (vn[c] + vm[c] + h * a[c]);
    }
}

/*
 * One group: q, v [n][3] in/out (body-major), m [n], rc [nlevels][n].
 * stats (if not NULL): [0] accepted macro steps, [1] rejected (halved) attempts, [2] force evaluations.
 * returns 0, or 1 if a macro step did not converge after BS_MAX_HALVINGS halvings (state left at the last
 * accepted time).
 */
int genga_oracle_bs_group_tp(int32_t n, int32_t nlevels, double G, double m_star, double dt, double tol,
                             const double *m, const double *rc, double *q, double *v, int64_t *stats,
                             const int8_t *is_tp, int32_t tp_mode)
{
    bs_group g = {n, nlevels, G, G * m_star, m, rc, is_tp, tp_mode};
    const int n3 = 3 * n;
    /* P[j] holds T_{k-1,j} of the previous row, component-wise: Pq[j][n3], Pv[j][n3] */
    double *buf = (double *)malloc((size_t)(2 * BS_KMAX * n3 + 5 * n3 + 5 * n3) * sizeof(double));
    double *Pq = buf, *Pv = buf + BS_KMAX * n3;
    double *cq = buf + 2 * BS_KMAX * n3, *cv = cq + n3, *a0 = cv + n3, *dq = a0 + n3, *dv = dq + n3, *w = dv + n3;
    int64_t acc = 0, rej = 0, fev = 0;
    double done = 0.0, H = dt;
    int fail = 0;
    while (done != dt) {
        if ((dt > 0.0 && done + H > dt) || (dt < 0.0 && done + H < dt)) H = dt - done;
        bs_accel(&g, q, a0); fev++;
        int halvings = 0, kconv = 0;
        for (;;) {
            int ok = 0;
            for (int k = 0; k < BS_KMAX; k++) {
                const int nk = 2 * (k + 1);
                bs_midpoint(&g, q, v, a0, H, nk, cq, cv, w); fev += nk;       /* cur = T_{k,0} */
                for (int j = 1; j <= k; j++) {
                    const double ratio = (double)nk / (double)(2 * (k - j + 1));   /* n_k / n_{k-j} */
                    const double den = ratio * ratio - 1.0;
                    for (int c = 0; c < n3; c++) {
                        const double lq = cq[c], lv = cv[c];                       /* T_{k,j-1} */
                        const double nq = lq + (lq - Pq[(j - 1) * n3 + c]) / den;  /* T_{k,j}   */
                        const double nv = lv + (lv - Pv[(j - 1) * n3 + c]) / den;
                        Pq[(j - 1) * n3 + c] = lq; Pv[(j - 1) * n3 + c] = lv;
                        cq[c] = nq; cv[c] = nv;
                        dq[c] = nq - lq; dv[c] = nv - lv;                          /* after j = k: T_kk - T_k,k-1 */
                    }
                }
                for (int c = 0; c < n3; c++) { Pq[k * n3 + c] = cq[c]; Pv[k * n3 + c] = cv[c]; }   /* T_kk */
                if (k > 0) {
                    double errmax = 0.0;
                    for (int i = 0; i < n; i++) {
                        double eq2 = 0.0, sq2 = 0.0, ev2 = 0.0, sv2 = 0.0;
                        for (int c = 3 * i; c < 3 * i + 3; c++) {
                            eq2 = eq2 + dq[c] * dq[c]; sq2 = sq2 + cq[c] * cq[c];
                            ev2 = ev2 + dv[c] * dv[c]; sv2 = sv2 + cv[c] * cv[c];
                        }
                        const double eq = sqrt(eq2) / sqrt(sq2), ev = sqrt(ev2) / sqrt(sv2);
                        if (eq > errmax) errmax = eq;
                        if (ev > errmax) errmax = ev;
                    }
                    if (errmax <= tol) { ok = 1; kconv = k + 1; break; }
                }
            }
            if (ok) break;
            rej++;
            if (++halvings > BS_MAX_HALVINGS) { fail = 1; break; }
            H = 0.5 * H;
        }
        if (fail) break;
        for (int c = 0; c < n3; c++) { q[c] = cq[c]; v[c] = cv[c]; }
        acc++;
        if ((dt > 0.0 && done + H >= dt) || (dt < 0.0 && done + H <= dt)) done = dt;
        else done = done + H;
        if (kconv <= 5) H = 2.0 * H;
    }
    if (stats) { stats[0] = acc; stats[1] = rej; stats[2] = fev; }
    free(buf);
    return fail;
}

/* fully interactive group (TP 0) */
int genga_oracle_bs_group(int32_t n, int32_t nlevels, double G, double m_star, double dt, double tol,
                          const double *m, const double *rc, double *q, double *v, int64_t *stats)
{
    return genga_oracle_bs_group_tp(n, nlevels, G, m_star, dt, tol, m, rc, q, v, stats, 0, 0);
}
