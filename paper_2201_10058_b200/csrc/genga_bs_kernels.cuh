// sm_100a kernel of the Bulirsch-Stoer integration of close-encounter groups (include/genga_bs.h;
// PAPER.md:47, :559-597, App. A).  One CTA per group, up to four bodies per thread (the regimes BS-B and
// BS-A of Table 2, and a little beyond: groups of up to 1024 bodies are integrated inside a
// single thread block through shared memory, with no host round trip between sub-steps).  Larger groups (the paper's BS-M,
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

#define GENGA_BS_THREADS 256
#define GENGA_BS_BPT 4                  // bodies per thread: groups of up to GENGA_BS_THREADS * GENGA_BS_BPT bodies
#define GENGA_BS_MAX_GROUP (GENGA_BS_THREADS * GENGA_BS_BPT)
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

// dynamic shared memory of bs_kernel: the group's positions, G m and critical radii, body-indexed
struct BsShared {
    double* x; double* y; double* z; double* gm;
    double* rc[GENGA_BS_MAX_LEVELS];
};
__host__ __device__ constexpr size_t bs_smem_bytes() { return (size_t)(4 + GENGA_BS_MAX_LEVELS) * GENGA_BS_MAX_GROUP * sizeof(double); }

// dv/dt of body i at the positions the group has published in shared memory:
//   - G m_star q / |q|^3 + sum_{j != i} G m_j prod_k (1 - K(r; max(rc_k,i, rc_k,j))) (q_j - q) / r^3
__device__ __forceinline__ void bs_accel(const BsShared& S, int i, int n, int nlevels, double mu, double x, double y,
                                         double z, double& ax, double& ay, double& az)
{
    const double r2s = x * x + y * y + z * z;
    const double rs = sqrt(r2s);
    const double s0 = -mu / (r2s * rs);
    ax = s0 * x; ay = s0 * y; az = s0 * z;
    for (int j = 0; j < n; j++) {
        if (j == i) continue;
        const double dx = S.x[j] - x, dy = S.y[j] - y, dz = S.z[j] - z;
        const double r2 = dx * dx + dy * dy + dz * dz;
        const double r = sqrt(r2);
        double W = 1.0;
        for (int k = 0; k < nlevels; k++) W *= (1.0 - bs_K(r, fmax(S.rc[k][i], S.rc[k][j])));
        if (W != 0.0) {
            const double s = S.gm[j] * W / (r2 * r);
            ax = ax + s * dx; ay = ay + s * dy; az = az + s * dz;
        }
    }
}

// every thread publishes the positions of its bodies (i = t + u * GENGA_BS_THREADS < n) and gets their accelerations
__device__ __forceinline__ void bs_force(const BsShared& S, int t, int n, int nlevels, double mu,
                                         const double (&q)[GENGA_BS_BPT][3], double (&a)[GENGA_BS_BPT][3])
{
    __syncthreads();                                          // the previous readers are done
#pragma unroll
    for (int u = 0; u < GENGA_BS_BPT; u++) {
        const int i = t + u * GENGA_BS_THREADS;
        if (i < n) { S.x[i] = q[u][0]; S.y[i] = q[u][1]; S.z[i] = q[u][2]; }
    }
    __syncthreads();
#pragma unroll
    for (int u = 0; u < GENGA_BS_BPT; u++) {
        const int i = t + u * GENGA_BS_THREADS;
        if (i < n) bs_accel(S, i, n, nlevels, mu, q[u][0], q[u][1], q[u][2], a[u][0], a[u][1], a[u][2]);
    }
}

__global__ void __launch_bounds__(GENGA_BS_THREADS)
bs_kernel(const double* __restrict__ pos_in, const double* __restrict__ vel_in, const double* __restrict__ mass,
          const double* __restrict__ rcrit, long long N, int nlevels, double G, double mu, double dt, double tol,
          const int* __restrict__ members, const int* __restrict__ offsets, const int* __restrict__ summary,
          double* __restrict__ pos, double* __restrict__ vel, int* __restrict__ status)
{
    constexpr int BPT = GENGA_BS_BPT;
    extern __shared__ __align__(16) double bs_smem[];
    __shared__ double red[GENGA_BS_THREADS / 32];
    __shared__ double errmax;
    BsShared S;
    S.x = bs_smem; S.y = S.x + GENGA_BS_MAX_GROUP; S.z = S.y + GENGA_BS_MAX_GROUP; S.gm = S.z + GENGA_BS_MAX_GROUP;
#pragma unroll
    for (int k = 0; k < GENGA_BS_MAX_LEVELS; k++) S.rc[k] = S.gm + (size_t)(k + 1) * GENGA_BS_MAX_GROUP;
    const int t = threadIdx.x;
    const int n_groups = summary[0];
    for (int g = blockIdx.x; g < n_groups; g += gridDim.x) {
        const int first = offsets[g], n = offsets[g + 1] - first;
        if (n > GENGA_BS_MAX_GROUP) {                          // CTA-uniform
            if (t == 0) atomicOr(status, GENGA_STATUS_GROUP_TOO_LARGE);
            continue;
        }
        long long b[BPT];
        double q[BPT][3], v[BPT][3];
        __syncthreads();                                      // the previous group's readers are done
#pragma unroll
        for (int u = 0; u < BPT; u++) {
            const int i = t + u * GENGA_BS_THREADS;
            b[u] = 0;
#pragma unroll
            for (int c = 0; c < 3; c++) { q[u][c] = 0.0; v[u][c] = 0.0; }
            if (i < n) {
                b[u] = members[first + i];
#pragma unroll
                for (int c = 0; c < 3; c++) { q[u][c] = pos_in[c * N + b[u]]; v[u][c] = vel_in[c * N + b[u]]; }
                S.gm[i] = G * mass[b[u]];
                for (int k = 0; k < nlevels; k++) S.rc[k][i] = rcrit[(long long)k * N + b[u]];
            }
        }
        double Pq[BPT][GENGA_BS_KMAX][3], Pv[BPT][GENGA_BS_KMAX][3];   // P[j] = T_{k-1,j} of the extrapolation tableau
        double a0[BPT][3], cq[BPT][3], cv[BPT][3], dq[BPT][3], dv[BPT][3];
        double done = 0.0, H = dt;
        bool fail = false;
        while (done != dt) {                                  // all decisions below are CTA-uniform
            if ((dt > 0.0 && done + H > dt) || (dt < 0.0 && done + H < dt)) H = dt - done;
            bs_force(S, t, n, nlevels, mu, q, a0);
            int halvings = 0, kconv = 0;
            for (;;) {
                bool ok = false;
                for (int k = 0; k < GENGA_BS_KMAX; k++) {
                    const int nk = 2 * (k + 1);
                    {   // modified midpoint over H with nk sub-steps: (q, v) -> (cq, cv) = T_{k,0}
                        const double h = H / (double)nk, h2 = 2.0 * h;
                        double qm[BPT][3], vm[BPT][3], qn[BPT][3], vn[BPT][3], a[BPT][3];
#pragma unroll
                        for (int u = 0; u < BPT; u++)
#pragma unroll
                            for (int c = 0; c < 3; c++) {
                                qm[u][c] = q[u][c]; vm[u][c] = v[u][c];
                                qn[u][c] = q[u][c] + h * v[u][c]; vn[u][c] = v[u][c] + h * a0[u][c];
                                a[u][c] = 0.0;
                            }
                        for (int m = 1; m < nk; m++) {
                            bs_force(S, t, n, nlevels, mu, qn, a);
#pragma unroll
                            for (int u = 0; u < BPT; u++)
#pragma unroll
                                for (int c = 0; c < 3; c++) {
                                    const double qs = qm[u][c] + h2 * vn[u][c], vs = vm[u][c] + h2 * a[u][c];
                                    qm[u][c] = qn[u][c]; vm[u][c] = vn[u][c]; qn[u][c] = qs; vn[u][c] = vs;
                                }
                        }
                        bs_force(S, t, n, nlevels, mu, qn, a);
#pragma unroll
                        for (int u = 0; u < BPT; u++)
#pragma unroll
                            for (int c = 0; c < 3; c++) {
                                cq[u][c] = 0.5 * (qn[u][c] + qm[u][c] + h * vn[u][c]);
                                cv[u][c] = 0.5 * (vn[u][c] + vm[u][c] + h * a[u][c]);
                            }
                    }
                    for (int j = 1; j <= k; j++) {
                        const double ratio = (double)nk / (double)(2 * (k - j + 1));      // n_k / n_{k-j}
                        const double den = ratio * ratio - 1.0;
#pragma unroll
                        for (int u = 0; u < BPT; u++)
#pragma unroll
                            for (int c = 0; c < 3; c++) {
                                const double lq = cq[u][c], lv = cv[u][c];                // T_{k,j-1}
                                const double nq = lq + (lq - Pq[u][j - 1][c]) / den;      // T_{k,j}
                                const double nv = lv + (lv - Pv[u][j - 1][c]) / den;
                                Pq[u][j - 1][c] = lq; Pv[u][j - 1][c] = lv;
                                cq[u][c] = nq; cv[u][c] = nv;
                                dq[u][c] = nq - lq; dv[u][c] = nv - lv;                   // after j = k: T_kk - T_k,k-1
                            }
                    }
#pragma unroll
                    for (int u = 0; u < BPT; u++)
#pragma unroll
                        for (int c = 0; c < 3; c++) { Pq[u][k][c] = cq[u][c]; Pv[u][k][c] = cv[u][c]; }   // T_kk
                    if (k > 0) {
                        double e = 0.0;
#pragma unroll
                        for (int u = 0; u < BPT; u++) {
                            if (t + u * GENGA_BS_THREADS >= n) continue;
                            double eq2 = 0.0, sq2 = 0.0, ev2 = 0.0, sv2 = 0.0;
#pragma unroll
                            for (int c = 0; c < 3; c++) {
                                eq2 = eq2 + dq[u][c] * dq[u][c]; sq2 = sq2 + cq[u][c] * cq[u][c];
                                ev2 = ev2 + dv[u][c] * dv[u][c]; sv2 = sv2 + cv[u][c] * cv[u][c];
                            }
                            e = fmax(e, fmax(sqrt(eq2) / sqrt(sq2), sqrt(ev2) / sqrt(sv2)));
                        }
                        // maximum over the group (order-free)
#pragma unroll
                        for (int o = 16; o > 0; o >>= 1) e = fmax(e, __shfl_xor_sync(0xffffffffu, e, o));
                        __syncthreads();
                        if ((t & 31) == 0) red[t >> 5] = e;
                        __syncthreads();
                        if (t == 0) {
                            double m = red[0];
#pragma unroll
                            for (int w = 1; w < GENGA_BS_THREADS / 32; w++) m = fmax(m, red[w]);
                            errmax = m;
                        }
                        __syncthreads();
                        if (errmax <= tol) { ok = true; kconv = k + 1; break; }
                    }
                }
                if (ok) break;
                if (++halvings > GENGA_BS_MAX_HALVINGS) { fail = true; break; }
                H = 0.5 * H;
            }
            if (fail) break;
#pragma unroll
            for (int u = 0; u < BPT; u++)
#pragma unroll
                for (int c = 0; c < 3; c++) { q[u][c] = cq[u][c]; v[u][c] = cv[u][c]; }
            if ((dt > 0.0 && done + H >= dt) || (dt < 0.0 && done + H <= dt)) done = dt;
            else done = done + H;
            if (kconv <= 5) H = 2.0 * H;
        }
        if (fail && t == 0) atomicOr(status, GENGA_STATUS_BS_NOT_CONVERGED);
#pragma unroll
        for (int u = 0; u < BPT; u++)                          // (after a failure: the state at the last accepted time)
            if (t + u * GENGA_BS_THREADS < n) {
#pragma unroll
                for (int c = 0; c < 3; c++) { pos[c * N + b[u]] = q[u][c]; vel[c * N + b[u]] = v[u][c]; }
            }
    }
}

}  // namespace genga
