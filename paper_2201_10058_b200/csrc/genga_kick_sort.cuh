// Internal body order of the kick.
//
// The pair loop is fastest when a warp's i-bodies and a chunk's j-bodies are neighbours in space:
// then almost every (warp, chunk) combination is provably out of range of every critical radius
// and runs without any per-pair check.  The library therefore works on a spatially sorted copy
// of the bodies: key = class bit (massive / test particle) | 16-bit Hilbert-curve index of the
// (x, y) cell in a 256 x 256 grid over the bounding box.  The caller never sees this order (indices in
// the outputs are the caller's).
//
// The sort is a least-significant-digit radix sort (8 + 9 bits), STABLE, hence a fixed function
// of the inputs: the summation order, and with it every output bit, is reproducible from call to
// call ("reductions have a well defined order").  No atomics decide an order.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace genga {

#define GENGA_SORT_THREADS 256
// keys per sort CTA: 1024 up to 2^18 bodies (64 CTAs per pass at N = 65,536: blocks of 4096 left the SMs idle), 4096
// beyond (the single-CTA scan of digits x blocks counters is what grows with the number of blocks)
static inline int genga_sort_block(long long n) { return n > (1LL << 18) ? 4096 : 1024; }
#define GENGA_SORT_MAXDIGITS 512
#define GENGA_GRID_BITS 8

// order-preserving map float -> uint32 (for atomicMin / atomicMax)
__device__ __forceinline__ unsigned f2ord(float f)
{
    const unsigned u = __float_as_uint(f);
    return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__device__ __forceinline__ float ord2f(unsigned u)
{
    return __uint_as_float((u & 0x80000000u) ? (u & 0x7fffffffu) : ~u);
}

// bbox[0..3] = ord(min x), ord(min y), ord(max x), ord(max y)
static __global__ void sort_init_kernel(unsigned* __restrict__ bbox)
{
    if (threadIdx.x < 2) bbox[threadIdx.x] = 0xffffffffu;
    else if (threadIdx.x < 4) bbox[threadIdx.x] = 0u;
}

static __global__ void __launch_bounds__(256)
bbox_kernel(const double* __restrict__ pos, int N, unsigned* __restrict__ bbox)
{
    float lox = 3.0e38f, loy = 3.0e38f, hix = -3.0e38f, hiy = -3.0e38f;
    for (int b = blockIdx.x * blockDim.x + threadIdx.x; b < N; b += gridDim.x * blockDim.x) {
        const double x = pos[b], y = pos[(size_t)N + b];
        lox = fminf(lox, __double2float_rd(x)); hix = fmaxf(hix, __double2float_ru(x));
        loy = fminf(loy, __double2float_rd(y)); hiy = fmaxf(hiy, __double2float_ru(y));
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        lox = fminf(lox, __shfl_xor_sync(0xffffffffu, lox, o)); loy = fminf(loy, __shfl_xor_sync(0xffffffffu, loy, o));
        hix = fmaxf(hix, __shfl_xor_sync(0xffffffffu, hix, o)); hiy = fmaxf(hiy, __shfl_xor_sync(0xffffffffu, hiy, o));
    }
    if ((threadIdx.x & 31) == 0) {          // min / max do not depend on the order of the atomics
        atomicMin(bbox + 0, f2ord(lox)); atomicMin(bbox + 1, f2ord(loy));
        atomicMax(bbox + 2, f2ord(hix)); atomicMax(bbox + 3, f2ord(hiy));
    }
}

// Position of cell (x, y) of a 2^GENGA_GRID_BITS-square grid along the Hilbert curve.  Unlike the
// Morton (Z) order the curve never jumps: cells with consecutive indices share an edge, so any
// run of consecutive bodies is spatially compact -- which is what keeps the culling boxes small.
__device__ __forceinline__ unsigned hilbert_index(unsigned x, unsigned y)
{
    constexpr unsigned n = 1u << GENGA_GRID_BITS;
    unsigned d = 0;
#pragma unroll
    for (unsigned s = n >> 1; s > 0; s >>= 1) {
        const unsigned rx = (x & s) ? 1u : 0u, ry = (y & s) ? 1u : 0u;
        d += s * s * ((3u * rx) ^ ry);
        if (ry == 0) {                                        // rotate / reflect the quadrant
            if (rx) { x = (n - 1u) - x; y = (n - 1u) - y; }
            const unsigned t = x; x = y; y = t;
        }
    }
    return d;
}

// key of body b; counts of the first digit per sort block
static __global__ void __launch_bounds__(GENGA_SORT_THREADS)
key_hist_kernel(const double* __restrict__ pos, int N, int n_massive, const unsigned* __restrict__ bbox,
                unsigned* __restrict__ keys, int* __restrict__ vals, int bits, int n_blocks, int* __restrict__ counts, int block)
{
    __shared__ int hist[GENGA_SORT_MAXDIGITS];
    const int nd = 1 << bits;
    for (int d = threadIdx.x; d < nd; d += blockDim.x) hist[d] = 0;
    __syncthreads();
    const float x0 = ord2f(bbox[0]), y0 = ord2f(bbox[1]), x1 = ord2f(bbox[2]), y1 = ord2f(bbox[3]);
    const float cells = (float)(1 << GENGA_GRID_BITS);
    const float sx = x1 > x0 ? cells / (x1 - x0) : 0.0f, sy = y1 > y0 ? cells / (y1 - y0) : 0.0f;
    const int base = blockIdx.x * block;
    for (int q = threadIdx.x; q < block; q += blockDim.x) {
        const int b = base + q;
        if (b < N) {
            const float fx = ((float)pos[b] - x0) * sx, fy = ((float)pos[(size_t)N + b] - y0) * sy;
            // NaN or out-of-box values land in cell 0 / the last cell; any key gives a correct kick
            const unsigned ix = (unsigned)min(max((int)fx, 0), (1 << GENGA_GRID_BITS) - 1);
            const unsigned iy = (unsigned)min(max((int)fy, 0), (1 << GENGA_GRID_BITS) - 1);
            const unsigned key = (b >= n_massive ? 0x10000u : 0u) | hilbert_index(ix, iy);
            keys[b] = key;
            vals[b] = b;
            atomicAdd(&hist[key & (nd - 1)], 1);              // a count: order-free
        }
    }
    __syncthreads();
    for (int d = threadIdx.x; d < nd; d += blockDim.x) counts[(size_t)d * n_blocks + blockIdx.x] = hist[d];
}

static __global__ void __launch_bounds__(GENGA_SORT_THREADS)
radix_hist_kernel(const unsigned* __restrict__ keys, int N, int shift, int bits, int n_blocks, int* __restrict__ counts,
                  int block)
{
    __shared__ int hist[GENGA_SORT_MAXDIGITS];
    const int nd = 1 << bits;
    for (int d = threadIdx.x; d < nd; d += blockDim.x) hist[d] = 0;
    __syncthreads();
    const int base = blockIdx.x * block;
    for (int q = threadIdx.x; q < block; q += blockDim.x)
        if (base + q < N) atomicAdd(&hist[(keys[base + q] >> shift) & (nd - 1)], 1);
    __syncthreads();
    for (int d = threadIdx.x; d < nd; d += blockDim.x) counts[(size_t)d * n_blocks + blockIdx.x] = hist[d];
}

// exclusive prefix sum of counts[0..n) in place, one CTA, fixed order (integers: any order gives the same sums);
// four consecutive elements per thread and round (16-byte loads and stores when the array allows them)
static __global__ void __launch_bounds__(1024) scan_kernel(int* __restrict__ counts, int n)
{
    __shared__ int wsum[32];
    __shared__ int carry;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const bool vec = (n & 3) == 0 && (reinterpret_cast<uintptr_t>(counts) & 15u) == 0;
    for (int base = 0; base < n; base += 4096) {
        const int q = base + 4 * threadIdx.x;
        int e[4] = {0, 0, 0, 0};
        if (vec) {
            if (q < n) { const int4 v4 = *reinterpret_cast<const int4*>(counts + q); e[0] = v4.x; e[1] = v4.y; e[2] = v4.z; e[3] = v4.w; }
        } else {
#pragma unroll
            for (int k = 0; k < 4; k++)
                if (q + k < n) e[k] = counts[q + k];
        }
        const int v = e[0] + e[1] + e[2] + e[3];
        int s = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, s, o);
            if (lane >= o) s += t;
        }
        if (lane == 31) wsum[w] = s;
        __syncthreads();
        if (w == 0) {
            int t = wsum[lane];
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int u = __shfl_up_sync(0xffffffffu, t, o);
                if (lane >= o) t += u;
            }
            wsum[lane] = t;                                    // inclusive over warps
        }
        __syncthreads();
        const int before = carry + (w ? wsum[w - 1] : 0) + s - v;
        const int x0 = before, x1 = x0 + e[0], x2 = x1 + e[1], x3 = x2 + e[2];
        if (vec) {
            if (q < n) *reinterpret_cast<int4*>(counts + q) = make_int4(x0, x1, x2, x3);
        } else {
            if (q < n) counts[q] = x0;
            if (q + 1 < n) counts[q + 1] = x1;
            if (q + 2 < n) counts[q + 2] = x2;
            if (q + 3 < n) counts[q + 3] = x3;
        }
        __syncthreads();
        if (threadIdx.x == 1023) carry = before + v;
        __syncthreads();
    }
}

// Stable scatter of one radix pass.  Warp w of a block owns the block's items
// [w * 512, (w + 1) * 512) and walks them in order, 32 at a time; the rank of an item among the
// items of the same digit is (global offset of digit, block) + (count in lower warps) + (count in
// earlier rounds of this warp) + (lower lanes of this round): no atomics, input order kept.
static __global__ void __launch_bounds__(GENGA_SORT_THREADS)
radix_scatter_kernel(const unsigned* __restrict__ keys_in, const int* __restrict__ vals_in, int N, int shift, int bits,
                     int n_blocks, const int* __restrict__ offsets, unsigned* __restrict__ keys_out,
                     int* __restrict__ vals_out, int block)
{
    constexpr int WARPS = GENGA_SORT_THREADS / 32;
    const int PER_WARP = block / WARPS;
    __shared__ int whist[WARPS][GENGA_SORT_MAXDIGITS];
    const int nd = 1 << bits;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    for (int d = threadIdx.x; d < WARPS * GENGA_SORT_MAXDIGITS; d += blockDim.x) (&whist[0][0])[d] = 0;
    __syncthreads();
    const int wbase = blockIdx.x * block + w * PER_WARP;
    for (int r = 0; r < PER_WARP; r += 32) {
        const int q = wbase + r + lane;
        if (q < N) atomicAdd(&whist[w][(keys_in[q] >> shift) & (nd - 1)], 1);    // a count: order-free
    }
    __syncthreads();
    for (int d = threadIdx.x; d < nd; d += blockDim.x) {
        int run = offsets[(size_t)d * n_blocks + blockIdx.x];
#pragma unroll
        for (int v = 0; v < WARPS; v++) {
            const int c = whist[v][d];
            whist[v][d] = run;
            run += c;
        }
    }
    __syncthreads();
    for (int r = 0; r < PER_WARP; r += 32) {
        const int q = wbase + r + lane;
        const bool live = q < N;
        const unsigned key = live ? keys_in[q] : 0u;
        const int d = live ? (int)((key >> shift) & (nd - 1)) : nd;          // nd: no real digit
        const unsigned peers = __match_any_sync(0xffffffffu, d);
        if (live) {
            const int slot = whist[w][d] + __popc(peers & ((1u << lane) - 1u));
            if (keys_out) keys_out[slot] = key;
            vals_out[slot] = vals_in[q];
        }
        __syncwarp();
        if (live && lane == __ffs(peers) - 1) whist[w][d] += __popc(peers);
        __syncwarp();
    }
}

}  // namespace genga
