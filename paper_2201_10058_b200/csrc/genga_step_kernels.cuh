// sm_100a kernels of the O(N) neighbours of the kick (include/genga_step.h): Rcrit (eq. 5
// PAPER.md:72-76, :638), HC (eq. 4), FG (Kepler part of eq. 2), as they
// appear in the step of App. A.  All of them are HBM/latency-bound passes over
// 56-64 bytes per body; what matters is the number of launches and a FIXED summation order.
//
// Work decomposition shared by every kernel here (so that the fused drift kernel adds the momenta
// in exactly the order psum_kernel does): nb = step_blocks(N) CTAs of GENGA_STEP_THREADS threads;
// CTA b owns the bodies [b * chunk, (b + 1) * chunk), chunk = step_chunk(N) (a multiple of the CTA
// size); thread t visits b * chunk + t + k * GENGA_STEP_THREADS for k = 0, 1, ... in that order.
//
// No code, header, table or helper is shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace genga {

#define GENGA_STEP_THREADS 256
#define GENGA_PSUM_BLOCKS 1024          // most CTAs of a step kernel = rows of the partial-sum scratch
#define GENGA_STATUS_UNBOUND 8
#define GENGA_STATUS_BAD_INDEX 16       // an index of a body list outside [0, N): entry ignored

__host__ __device__ __forceinline__ int step_blocks(long long N)
{
    const long long nb = (N + GENGA_STEP_THREADS - 1) / GENGA_STEP_THREADS;
    return (int)(nb < GENGA_PSUM_BLOCKS ? (nb > 0 ? nb : 1) : GENGA_PSUM_BLOCKS);
}
__host__ __device__ __forceinline__ long long step_chunk(long long N)
{
    const long long nb = step_blocks(N);
    const long long per = (N + nb - 1) / nb;
    return (per + GENGA_STEP_THREADS - 1) / GENGA_STEP_THREADS * GENGA_STEP_THREADS;
}

// ---------------------------------------------------------------------------------------------
// Rcrit (eq. 5): out[k][i] = max(n1 R_H,i, n2 (dt / s^k) |v_i|), R_H,i = a_i (m_i / 3 m_star)^(1/3),
// 1/a_i = 2/r - v^2/mu (vis-viva, mu = G m_star).
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(GENGA_STEP_THREADS)
rcrit_kernel(const double* __restrict__ pos, const double* __restrict__ vel, const double* __restrict__ mass,
             long long N, double mu, double m_star, double dt, double substeps, int nrows, double n1, double n2,
             double* __restrict__ out, int* __restrict__ status, const int* __restrict__ list,
             const int* __restrict__ n_list, long long list_rows)
{
    // list == nullptr: every body; else the bodies list[0 .. min(*n_list, list_rows)) ("RcritS", App. A)
    const long long count = list ? min((long long)max(*n_list, 0), list_rows) : N;
    for (long long q = (long long)blockIdx.x * GENGA_STEP_THREADS + threadIdx.x; q < count;
         q += (long long)gridDim.x * GENGA_STEP_THREADS) {
        const long long i = list ? list[q] : q;
        if (i < 0 || i >= N) { atomicOr(status, GENGA_STATUS_BAD_INDEX); continue; }
        const double x = pos[i], y = pos[N + i], z = pos[2 * N + i];
        const double vx = vel[i], vy = vel[N + i], vz = vel[2 * N + i];
        const double r = sqrt(fma(z, z, fma(y, y, x * x)));
        const double v2 = fma(vz, vz, fma(vy, vy, vx * vx));
        const double inv_a = 2.0 / r - v2 / mu;
        double hill = 0.0;
        if (inv_a > 0.0) hill = cbrt(mass[i] / (3.0 * m_star)) / inv_a;
        else atomicOr(status, GENGA_STATUS_UNBOUND);
        const double v = sqrt(v2);
        const double a = n1 * hill;
        double dtk = dt;
        for (int k = 0; k < nrows; k++) {
            out[(long long)k * N + i] = fmax(a, n2 * dtk * v);
            dtk /= substeps;
        }
    }
}

// ---------------------------------------------------------------------------------------------
// Fixed-order sum of the CTA's three per-thread values: xor-butterfly inside each warp, then the
// warp sums in ascending warp order.  Returns the CTA sum in thread 0.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ void block_sum3(double& a, double& b, double& c)
{
    __shared__ double sh[3][GENGA_STEP_THREADS / 32];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        a += __shfl_xor_sync(0xffffffffu, a, o);
        b += __shfl_xor_sync(0xffffffffu, b, o);
        c += __shfl_xor_sync(0xffffffffu, c, o);
    }
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (lane == 0) { sh[0][warp] = a; sh[1][warp] = b; sh[2][warp] = c; }
    __syncthreads();
    if (threadIdx.x == 0) {
        a = sh[0][0]; b = sh[1][0]; c = sh[2][0];
#pragma unroll
        for (int w = 1; w < GENGA_STEP_THREADS / 32; w++) { a += sh[0][w]; b += sh[1][w]; c += sh[2][w]; }
    }
}

// The CTA's partial sum goes to partial[blockIdx.x][3]; the CTA that finishes last (ticket) adds the
// partials -- thread t takes the CTAs t, t + 256, ... in ascending order, then the same fixed tree as
// above -- and writes the total to partial[GENGA_PSUM_BLOCKS + slot][3].  (A single thread adding up to
// 1024 partials one L2 round trip after the other took 20 us of the 22 us of psum_kernel.)
__device__ __forceinline__ void publish_sum3(double a, double b, double c, double* __restrict__ partial,
                                             unsigned* __restrict__ ticket, int slot)
{
    __shared__ bool last;
    if (threadIdx.x == 0) {
        partial[3 * blockIdx.x + 0] = a; partial[3 * blockIdx.x + 1] = b; partial[3 * blockIdx.x + 2] = c;
        __threadfence();
        last = atomicAdd(ticket, 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (!last) return;                                       // CTA-uniform
    __threadfence();
    double ta = 0.0, tb = 0.0, tc = 0.0;
    for (unsigned q = threadIdx.x; q < gridDim.x; q += GENGA_STEP_THREADS) {
        ta += __ldcg(partial + 3 * q + 0); tb += __ldcg(partial + 3 * q + 1); tc += __ldcg(partial + 3 * q + 2);
    }
    __syncthreads();                                         // block_sum3's shared array is reused
    block_sum3(ta, tb, tc);
    if (threadIdx.x == 0) {
        double* tot = partial + 3 * (GENGA_PSUM_BLOCKS + slot);
        tot[0] = ta; tot[1] = tb; tot[2] = tc;
        *ticket = 0u;                                        // ready for the next launch on the stream
    }
}

// sum_j m_j v_j  ->  partial[GENGA_PSUM_BLOCKS + slot][3]
__global__ void __launch_bounds__(GENGA_STEP_THREADS)
psum_kernel(const double* __restrict__ vel, const double* __restrict__ mass, long long N,
            double* __restrict__ partial, unsigned* __restrict__ ticket, int slot)
{
    const long long chunk = step_chunk(N), base = (long long)blockIdx.x * chunk;
    double px = 0.0, py = 0.0, pz = 0.0;
    for (long long i = base + threadIdx.x; i < base + chunk && i < N; i += GENGA_STEP_THREADS) {
        const double m = mass[i];
        px = fma(m, vel[i], px); py = fma(m, vel[N + i], py); pz = fma(m, vel[2 * N + i], pz);
    }
    block_sum3(px, py, pz);
    publish_sum3(px, py, pz, partial, ticket, slot);
}

// HC (eq. 4): pos_i += (dt * P) / m_star with P = partial[GENGA_PSUM_BLOCKS + slot]
__global__ void __launch_bounds__(GENGA_STEP_THREADS)
shift_kernel(double* __restrict__ pos, long long N, const double* __restrict__ partial, int slot, double dt, double m_star)
{
    const double* P = partial + 3 * (GENGA_PSUM_BLOCKS + slot);
    const double sx = dt * P[0] / m_star, sy = dt * P[1] / m_star, sz = dt * P[2] / m_star;
    const long long chunk = step_chunk(N), base = (long long)blockIdx.x * chunk;
    for (long long i = base + threadIdx.x; i < base + chunk && i < N; i += GENGA_STEP_THREADS) {
        pos[i] += sx; pos[N + i] += sy; pos[2 * N + i] += sz;
    }
}

// ---------------------------------------------------------------------------------------------
// FG: the exact two-body motion over dt with Gauss' f and g functions in the difference dE of the
// eccentric anomaly.  Kepler's equation in difference form,
//     F(dE) = dE - ec sin dE + es (1 - cos dE) - dM = 0,   ec = e cos E0 = 1 - r0/a,  es = e sin E0 = u / (n a^2),
// has F' = r/a > 0: F is increasing and |F(dE) - (dE - dM)| <= |ec| + 2 |es|, so the root lies in
// dM +- (|ec| + 2 |es|); Newton from dE = dM, any step that leaves the bracket replaced by its
// midpoint (bisection), which converges for every bound orbit.
// A hyperbolic orbit (1/a < 0: an ejected body, or one above the escape speed inside a deep passage) takes the same
// two-body solution in the difference dH of the hyperbolic anomaly, with a' = -a, n' = sqrt(mu / a'^3):
//     F(dH) = ec sinh dH + es (cosh dH - 1) - dH - n' dt = 0,   ec = 1 + r0/a',  es = u / (n' a'^2),   F' = r/a' > 0,
// bracketed by doubling from 0, then the same safeguarded Newton iteration.
// Returns false (state untouched) only for 1/a = 0 exactly (parabolic) or a state that is not a number.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ bool kepler_fg(double mu, double dt, double& x, double& y, double& z,
                                          double& vx, double& vy, double& vz)
{
    const double r0 = sqrt(fma(z, z, fma(y, y, x * x)));
    const double v2 = fma(vz, vz, fma(vy, vy, vx * vx));
    const double u = fma(z, vz, fma(y, vy, x * vx));
    const double inv_a = 2.0 / r0 - v2 / mu;
    if (inv_a < 0.0) {
        const double ap = -1.0 / inv_a;
        const double np_ = sqrt(-mu * inv_a) * -inv_a;       // sqrt(mu / a'^3)
        const double ec = 1.0 + r0 / ap, es = u / (np_ * ap * ap), dN = np_ * dt;
        double lo = 0.0, hi = 0.0, w = 1.0;
        for (int it = 0; it < 64; it++) {                    // F is increasing and F(0) = -dN: the root lies beyond 0 on dN's side
            const double xw = dN > 0.0 ? w : -w;
            const double fn = ec * sinh(xw) + es * (cosh(xw) - 1.0) - xw - dN;
            if (dN > 0.0 ? fn >= 0.0 : fn <= 0.0) { if (dN > 0.0) hi = xw; else lo = xw; break; }
            if (dN > 0.0) lo = xw; else hi = xw;
            w *= 2.0;
        }
        double dH = 0.5 * (lo + hi), sh, ch;
        for (int it = 0; it < 80; it++) {
            sh = sinh(dH); ch = cosh(dH);
            const double fn = ec * sh + es * (ch - 1.0) - dH - dN;
            const double fp = ec * ch + es * sh - 1.0;
            if (fn > 0.0) hi = dH; else lo = dH;
            double nx = dH - fn / fp;
            if (!(nx > lo && nx < hi)) nx = 0.5 * (lo + hi);
            const double step = nx - dH;
            dH = nx;
            if (fabs(step) <= 4.0e-16 * (1.0 + fabs(dH))) break;
        }
        sh = sinh(dH); ch = cosh(dH);
        const double r = ap * (ec * ch + es * sh - 1.0);
        const double f = 1.0 - (ap / r0) * (ch - 1.0);
        const double g = dt - (sh - dH) / np_;
        const double fd = -(ap * ap * np_ / (r0 * r)) * sh;
        const double gd = 1.0 - (ap / r) * (ch - 1.0);
        const double nx = f * x + g * vx, ny = f * y + g * vy, nz = f * z + g * vz;
        const double nvx = fd * x + gd * vx, nvy = fd * y + gd * vy, nvz = fd * z + gd * vz;
        x = nx; y = ny; z = nz; vx = nvx; vy = nvy; vz = nvz;
        return true;
    }
    if (!(inv_a > 0.0)) return false;
    const double a = 1.0 / inv_a;
    const double n = sqrt(mu * inv_a) * inv_a;               // mean motion sqrt(mu / a^3)
    const double ec = 1.0 - r0 * inv_a;
    const double es = u * inv_a * inv_a / n;
    const double dM = n * dt;
    const double w = fabs(ec) + 2.0 * fabs(es) + 1.0e-300;
    double lo = dM - w, hi = dM + w, dE = dM, s, c;
    for (int it = 0; it < 80; it++) {
        sincos(dE, &s, &c);
        const double fn = (dE - dM) - ec * s + es * (1.0 - c);
        const double fp = 1.0 - ec * c + es * s;
        if (fn > 0.0) hi = dE; else lo = dE;
        double nx = dE - fn / fp;
        if (!(nx > lo && nx < hi)) nx = 0.5 * (lo + hi);
        const double step = nx - dE;
        dE = nx;
        if (fabs(step) <= 4.0e-16 * (1.0 + fabs(dE))) break;
    }
    sincos(dE, &s, &c);
    const double omc = 1.0 - c;
    const double r = a * (1.0 - ec * c + es * s);
    const double f = 1.0 - (a / r0) * omc;
    const double g = dt + (s - dE) / n;
    const double fd = -(a * a * n / (r0 * r)) * s;
    const double gd = 1.0 - (a / r) * omc;
    const double nx = f * x + g * vx, ny = f * y + g * vy, nz = f * z + g * vz;
    const double nvx = fd * x + gd * vx, nvy = fd * y + gd * vy, nvz = fd * z + gd * vz;
    x = nx; y = ny; z = nz; vx = nvx; vy = nvy; vz = nvz;
    return true;
}

// FG alone (SHIFT = false, mass = partial = nullptr), or the middle of genga_drift (SHIFT = true):
//   pos_i += (h * P_in) / m_star  [HC(dt/2) with the momentum sum of slot_in];  FG(dt);
//   sum_j m_j v_j of the NEW velocities -> slot_out  [for the closing HC(dt/2)]
template <bool SHIFT>
__global__ void __launch_bounds__(GENGA_STEP_THREADS)
fg_kernel(double* __restrict__ pos, double* __restrict__ vel, const double* __restrict__ mass, long long N, double mu,
          double dt, double h, double m_star, double* __restrict__ partial, unsigned* __restrict__ ticket,
          int slot_in, int slot_out, int* __restrict__ status)
{
    double sx = 0.0, sy = 0.0, sz = 0.0;
    if (SHIFT) {
        const double* P = partial + 3 * (GENGA_PSUM_BLOCKS + slot_in);
        sx = h * P[0] / m_star; sy = h * P[1] / m_star; sz = h * P[2] / m_star;
    }
    const long long chunk = step_chunk(N), base = (long long)blockIdx.x * chunk;
    double px = 0.0, py = 0.0, pz = 0.0;
    for (long long i = base + threadIdx.x; i < base + chunk && i < N; i += GENGA_STEP_THREADS) {
        double x = pos[i], y = pos[N + i], z = pos[2 * N + i];
        double vx = vel[i], vy = vel[N + i], vz = vel[2 * N + i];
        if (SHIFT) { x += sx; y += sy; z += sz; }
        if (!kepler_fg(mu, dt, x, y, z, vx, vy, vz)) atomicOr(status, GENGA_STATUS_UNBOUND);
        pos[i] = x; pos[N + i] = y; pos[2 * N + i] = z;
        vel[i] = vx; vel[N + i] = vy; vel[2 * N + i] = vz;
        if (SHIFT) {
            const double m = mass[i];
            px = fma(m, vx, px); py = fma(m, vy, py); pz = fma(m, vz, pz);
        }
    }
    if (SHIFT) {
        block_sum3(px, py, pz);
        publish_sum3(px, py, pz, partial, ticket, slot_out);
    }
}

// "FGS" (App. A): the Kepler drift of the bodies of a list only
__global__ void __launch_bounds__(GENGA_STEP_THREADS)
fg_list_kernel(double* __restrict__ pos, double* __restrict__ vel, long long N, double mu, double dt,
               const int* __restrict__ list, const int* __restrict__ n_list, long long list_rows, int* __restrict__ status)
{
    const long long count = min((long long)max(*n_list, 0), list_rows);
    for (long long q = (long long)blockIdx.x * GENGA_STEP_THREADS + threadIdx.x; q < count;
         q += (long long)gridDim.x * GENGA_STEP_THREADS) {
        const long long i = list[q];
        if (i < 0 || i >= N) { atomicOr(status, GENGA_STATUS_BAD_INDEX); continue; }
        double x = pos[i], y = pos[N + i], z = pos[2 * N + i];
        double vx = vel[i], vy = vel[N + i], vz = vel[2 * N + i];
        if (!kepler_fg(mu, dt, x, y, z, vx, vy, vz)) atomicOr(status, GENGA_STATUS_UNBOUND);
        pos[i] = x; pos[N + i] = y; pos[2 * N + i] = z;
        vel[i] = vx; vel[N + i] = vy; vel[2 * N + i] = vz;
    }
}

}  // namespace genga
