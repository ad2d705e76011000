// sm_100a kernel of the Bulirsch-Stoer integration of close-encounter groups (include/genga_bs.h;
// PAPER.md:47, :559-597, App. A).  One CTA per group, one thread per body (the regimes BS-B and
// BS-A of Table 2: groups of up to 256 bodies are integrated inside a single thread block
// through shared memory, with no host round trip between sub-steps).  Larger groups (the paper's BS-M,
// host-controlled sub-steps over several blocks) are not integrated: they are reported.
//
// The scheme is the textbook Gragg-Bulirsch-Stoer method fixed as reading G15 in DESIGN.md: modified
// midpoint with n_k = 2k sub-steps (k = 1..8), Aitken-Neville extrapolation in h^2, relative error per body
// (Euclidean norms of position and of velocity), the whole group advancing synchronously with one step
// size.  Every operation is written in the order of that description and the build forbids contraction
// (--fmad=false), the force sum runs over the group's members in list order: the result is a fixed
// function of the inputs.
//
// No code, header, table or helper is shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace genga {

#define GENGA_BS_THREADS 256            // = largest group integrated
#define GENGA_BS_KMAX 8
#define GENGA_BS_MAX_LEVELS 4
#define GENGA_BS_MAX_HALVINGS 60
#define GENGA_STATUS_GROUP_TOO_LARGE 32
#define GENGA_STATUS_BS_NOT_CONVERGED 64

// the changeover function K (reading G1), IEEE operations in a fixed order
__device__ __forceinline__ double bs_K(double r, double rc)
{
    const double y = (r - 0.1 * rc) / (0.9 * rc);
    if (y <= 0.0) return 0.0;
    if (y >= 1.0) return 1.0;
    return (y * y) / (2.0 * y * y - 2.0 * y + 1.0);
}

struct BsShared {
    double x[GENGA_BS_THREADS], y[GENGA_BS_THREADS], z[GENGA_BS_THREADS];
    double gm[GENGA_BS_THREADS];                              // G m_j
    double rc[GENGA_BS_MAX_LEVELS][GENGA_BS_THREADS];
    double red[GENGA_BS_THREADS / 32];
    double errmax;
};

// dv/dt of body t at the positions the group has published in shared memory:
//   - G m_star q / |q|^3 + sum_{j != t} G m_j prod_k (1 - K(r; max(rc_k,t, rc_k,j))) (q_j - q) / r^3
__device__ __forceinline__ void bs_accel(const BsShared& S, int t, int n, int nlevels, double mu, double x, double y,
                                         double z, double& ax, double& ay, double& az)
{
    const double r2s = x * x + y * y + z * z;
    const double rs = sqrt(r2s);
    const double s0 = -mu / (r2s * rs);
    ax = s0 * x; ay = s0 * y; az = s0 * z;
    for (int j = 0; j < n; j++) {
        if (j == t) continue;
        const double dx = S.x[j] - x, dy = S.y[j] - y, dz = S.z[j] - z;
        const double r2 = dx * dx + dy * dy + dz * dz;
        const double r = sqrt(r2);
        double W = 1.0;
        for (int k = 0; k < nlevels; k++) W *= (1.0 - bs_K(r, fmax(S.rc[k][t], S.rc[k][j])));
        if (W != 0.0) {
            const double s = S.gm[j] * W / (r2 * r);
            ax = ax + s * dx; ay = ay + s * dy; az = az + s * dz;
        }
    }
}

// every thread of the CTA publishes (x, y, z) and gets its acceleration back
__device__ __forceinline__ void bs_force(BsShared& S, bool active, int t, int n, int nlevels, double mu, const double (&q)[3],
                                         double (&a)[3])
{
    __syncthreads();                                          // the previous readers are done
    if (active) { S.x[t] = q[0]; S.y[t] = q[1]; S.z[t] = q[2]; }
    __syncthreads();
    if (active) bs_accel(S, t, n, nlevels, mu, q[0], q[1], q[2], a[0], a[1], a[2]);
}

__global__ void __launch_bounds__(GENGA_BS_THREADS)
bs_kernel(const double* __restrict__ pos_in, const double* __restrict__ vel_in, const double* __restrict__ mass,
          const double* __restrict__ rcrit, long long N, int nlevels, double G, double mu, double dt, double tol,
          const int* __restrict__ members, const int* __restrict__ offsets, const int* __restrict__ summary,
          double* __restrict__ pos, double* __restrict__ vel, int* __restrict__ status)
{
    __shared__ BsShared S;
    const int t = threadIdx.x;
    const int n_groups = summary[0];
    for (int g = blockIdx.x; g < n_groups; g += gridDim.x) {
        const int first = offsets[g], n = offsets[g + 1] - first;
        if (n > GENGA_BS_THREADS) {                            // CTA-uniform
            if (t == 0) atomicOr(status, GENGA_STATUS_GROUP_TOO_LARGE);
            continue;
        }
        const bool active = t < n;
        const long long b = active ? members[first + t] : 0;
        double q[3] = {0.0, 0.0, 0.0}, v[3] = {0.0, 0.0, 0.0};
        __syncthreads();                                      // the previous group's readers are done
        if (active) {
            q[0] = pos_in[b]; q[1] = pos_in[N + b]; q[2] = pos_in[2 * N + b];
            v[0] = vel_in[b]; v[1] = vel_in[N + b]; v[2] = vel_in[2 * N + b];
            S.gm[t] = G * mass[b];
            for (int k = 0; k < nlevels; k++) S.rc[k][t] = rcrit[(long long)k * N + b];
        }
        double Pq[GENGA_BS_KMAX][3], Pv[GENGA_BS_KMAX][3];    // P[j] = T_{k-1,j} of the extrapolation tableau
        double a0[3], cq[3], cv[3], dq[3], dv[3];
        double done = 0.0, H = dt;
        bool fail = false;
        while (done != dt) {                                  // all decisions below are CTA-uniform
            if ((dt > 0.0 && done + H > dt) || (dt < 0.0 && done + H < dt)) H = dt - done;
            bs_force(S, active, t, n, nlevels, mu, q, a0);
            int halvings = 0, kconv = 0;
            for (;;) {
                bool ok = false;
                for (int k = 0; k < GENGA_BS_KMAX; k++) {
                    const int nk = 2 * (k + 1);
                    {   // modified midpoint over H with nk sub-steps: (q, v) -> (cq, cv) = T_{k,0}
                        const double h = H / (double)nk, h2 = 2.0 * h;
                        double qm[3], vm[3], qn[3], vn[3], a[3];
#pragma unroll
                        for (int c = 0; c < 3; c++) { qm[c] = q[c]; vm[c] = v[c]; qn[c] = q[c] + h * v[c]; vn[c] = v[c] + h * a0[c]; }
                        for (int m = 1; m < nk; m++) {
                            bs_force(S, active, t, n, nlevels, mu, qn, a);
#pragma unroll
                            for (int c = 0; c < 3; c++) {
                                const double qs = qm[c] + h2 * vn[c], vs = vm[c] + h2 * a[c];
                                qm[c] = qn[c]; vm[c] = vn[c]; qn[c] = qs; vn[c] = vs;
                            }
                        }
                        bs_force(S, active, t, n, nlevels, mu, qn, a);
#pragma unroll
                        for (int c = 0; c < 3; c++) {
                            cq[c] = 0.5 * (qn[c] + qm[c] + h * vn[c]);
                            cv[c] = 0.5 * (vn[c] + vm[c] + h * a[c]);
                        }
                    }
                    for (int j = 1; j <= k; j++) {
                        const double ratio = (double)nk / (double)(2 * (k - j + 1));      // n_k / n_{k-j}
                        const double den = ratio * ratio - 1.0;
#pragma unroll
                        for (int c = 0; c < 3; c++) {
                            const double lq = cq[c], lv = cv[c];                          // T_{k,j-1}
                            const double nq = lq + (lq - Pq[j - 1][c]) / den;             // T_{k,j}
                            const double nv = lv + (lv - Pv[j - 1][c]) / den;
                            Pq[j - 1][c] = lq; Pv[j - 1][c] = lv;
                            cq[c] = nq; cv[c] = nv;
                            dq[c] = nq - lq; dv[c] = nv - lv;                             // after j = k: T_kk - T_k,k-1
                        }
                    }
#pragma unroll
                    for (int c = 0; c < 3; c++) { Pq[k][c] = cq[c]; Pv[k][c] = cv[c]; }   // T_kk
                    if (k > 0) {
                        double e = 0.0;
                        if (active) {
                            double eq2 = 0.0, sq2 = 0.0, ev2 = 0.0, sv2 = 0.0;
#pragma unroll
                            for (int c = 0; c < 3; c++) {
                                eq2 = eq2 + dq[c] * dq[c]; sq2 = sq2 + cq[c] * cq[c];
                                ev2 = ev2 + dv[c] * dv[c]; sv2 = sv2 + cv[c] * cv[c];
                            }
                            e = fmax(sqrt(eq2) / sqrt(sq2), sqrt(ev2) / sqrt(sv2));
                        }
                        // maximum over the group (order-free)
#pragma unroll
                        for (int o = 16; o > 0; o >>= 1) e = fmax(e, __shfl_xor_sync(0xffffffffu, e, o));
                        __syncthreads();
                        if ((t & 31) == 0) S.red[t >> 5] = e;
                        __syncthreads();
                        if (t == 0) {
                            double m = S.red[0];
#pragma unroll
                            for (int w = 1; w < GENGA_BS_THREADS / 32; w++) m = fmax(m, S.red[w]);
                            S.errmax = m;
                        }
                        __syncthreads();
                        if (S.errmax <= tol) { ok = true; kconv = k + 1; break; }
                    }
                }
                if (ok) break;
                if (++halvings > GENGA_BS_MAX_HALVINGS) { fail = true; break; }
                H = 0.5 * H;
            }
            if (fail) break;
#pragma unroll
            for (int c = 0; c < 3; c++) { q[c] = cq[c]; v[c] = cv[c]; }
            if ((dt > 0.0 && done + H >= dt) || (dt < 0.0 && done + H <= dt)) done = dt;
            else done = done + H;
            if (kconv <= 5) H = 2.0 * H;
        }
        if (fail && t == 0) atomicOr(status, GENGA_STATUS_BS_NOT_CONVERGED);
        if (active) {                                          // (after a failure: the state at the last accepted time)
            pos[b] = q[0]; pos[N + b] = q[1]; pos[2 * N + b] = q[2];
            vel[b] = v[0]; vel[N + b] = v[1]; vel[2 * N + b] = v[2];
        }
    }
}

}  // namespace genga
