// sort.cuh — gal_plan_bind_obs: reorder a fixed observation set along a space-filling curve of the (u, v) plane.
//
// Why (a fit evaluates many models against ONE observation set): the sampler's gather
// touches four spectrum nodes per point.  In time-major order — the order of a measurement
// set — consecutive points lie on different baselines, far apart in the plane, so the 32 gathers of a warp go
// to 32 different cache lines and every one of them is an L2 round trip.  chi2 does not depend on the order of
// the points, so the plan keeps a private copy of (u, v, Re V_obs, Im V_obs, w) sorted by the Morton (Z-order)
// index of the point folded into the u >= 0 half plane (the fold the listing applies).  A
// rotation by any PA keeps neighbours neighbours, so a warp's cells then share a few lines that stay in L1.
//
// The sort is a plain least-significant-digit radix sort of (key, index) pairs, 8 bits per pass, written here
// (no library): per-tile digit histograms, one exclusive scan in digit-major order, and a STABLE scatter — thread
// t of a tile owns EPT consecutive elements and ranks them after all elements of threads < t with the same
// digit.  Stable passes make the result the unique order (key, original index): binding the same data twice
// gives the same permutation, so chi2 stays run-to-run bit-identical.  One-off cost at bind time.
#pragma once
#include "common.cuh"

namespace galb {

constexpr int SORT_NT = 256, SORT_EPT = 16, SORT_TILE = SORT_NT * SORT_EPT, SORT_STRIDE = 258;

__device__ __forceinline__ unsigned int morton_spread12(unsigned int x) {     // 12 bits -> every other bit of 24
    x &= 0xFFFu;
    x = (x | (x << 8)) & 0x00FF00FFu;
    x = (x | (x << 4)) & 0x0F0F0F0Fu;
    x = (x | (x << 2)) & 0x33333333u;
    x = (x | (x << 1)) & 0x55555555u;
    return x;
}

// key[k] = Morton index of the point folded to u >= 0 on a 4096 x 4096 grid over [0, rmax] x [-rmax, rmax]
template <typename T>
__global__ void __launch_bounds__(256) uv_key_kernel(const T* __restrict__ u, const T* __restrict__ v, long long M,
                                                     double inv_rmax, unsigned int* __restrict__ key,
                                                     unsigned int* __restrict__ idx) {
    for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k < M; k += (long long)gridDim.x * blockDim.x) {
        double a = (double)u[k], b = (double)v[k];
        if (a < 0.0 || (a == 0.0 && b < 0.0)) { a = -a; b = -b; }
        const double qa = fmin(fmax(a * inv_rmax, 0.0), 1.0) * 4095.0;
        const double qb = fmin(fmax(0.5 * (b * inv_rmax + 1.0), 0.0), 1.0) * 4095.0;
        key[k] = morton_spread12((unsigned int)qa) | (morton_spread12((unsigned int)qb) << 1);
        idx[k] = (unsigned int)k;
    }
}

// per-tile digit histogram, stored digit-major: hist[d * ntiles + tile]
static __global__ void __launch_bounds__(SORT_NT) radix_hist_kernel(const unsigned int* __restrict__ key, long long M, int shift,
                                                             unsigned int* __restrict__ hist, int ntiles) {
    __shared__ unsigned int h[256];
    h[threadIdx.x] = 0;
    __syncthreads();
    const long long base = (long long)blockIdx.x * SORT_TILE;
    for (int e = 0; e < SORT_EPT; ++e) {
        const long long k = base + e * SORT_NT + threadIdx.x;
        if (k < M) atomicAdd(&h[(key[k] >> shift) & 255u], 1u);
    }
    __syncthreads();
    hist[(long long)threadIdx.x * ntiles + blockIdx.x] = h[threadIdx.x];
}

// exclusive scan of n values in place, one CTA (n is a few hundred thousand at most)
static __global__ void __launch_bounds__(1024) scan_exclusive_kernel(unsigned int* __restrict__ a, long long n) {
    __shared__ unsigned int part[1024];
    const long long chunk = (n + 1023) / 1024;
    const long long lo = threadIdx.x * chunk, hi = lo + chunk < n ? lo + chunk : n;
    unsigned int s = 0;
    for (long long i = lo; i < hi; ++i) s += a[i];
    part[threadIdx.x] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned int run = 0;
        for (int i = 0; i < 1024; ++i) { const unsigned int t = part[i]; part[i] = run; run += t; }
    }
    __syncthreads();
    unsigned int run = part[threadIdx.x];
    for (long long i = lo; i < hi; ++i) { const unsigned int t = a[i]; a[i] = run; run += t; }
}

// stable scatter of one tile: thread t owns elements [t * EPT, (t + 1) * EPT) of the tile
static __global__ void __launch_bounds__(SORT_NT) radix_scatter_kernel(const unsigned int* __restrict__ key_in,
                                                                const unsigned int* __restrict__ idx_in, long long M,
                                                                int shift, const unsigned int* __restrict__ hist, int ntiles,
                                                                unsigned int* __restrict__ key_out,
                                                                unsigned int* __restrict__ idx_out) {
    extern __shared__ unsigned short cnt[];                  // [256 digits][SORT_STRIDE]: count, then prefix over threads
    const int t = threadIdx.x;
    for (int i = t; i < 256 * SORT_STRIDE; i += SORT_NT) cnt[i] = 0;
    __syncthreads();
    const long long base = (long long)blockIdx.x * SORT_TILE + (long long)t * SORT_EPT;
    unsigned int k[SORT_EPT], ix[SORT_EPT];
#pragma unroll
    for (int e = 0; e < SORT_EPT; ++e) {
        const long long p = base + e;
        k[e] = p < M ? key_in[p] : 0xFFFFFFFFu;
        ix[e] = p < M ? idx_in[p] : 0u;
        if (p < M) cnt[((k[e] >> shift) & 255u) * SORT_STRIDE + t] += 1;     // own column: no race
    }
    __syncthreads();
    {                                                        // thread d: exclusive prefix of digit d over the threads
        unsigned short* row = cnt + t * SORT_STRIDE;
        unsigned int run = 0;
        for (int i = 0; i < SORT_NT; ++i) { const unsigned int c = row[i]; row[i] = (unsigned short)run; run += c; }
    }
    __syncthreads();
#pragma unroll
    for (int e = 0; e < SORT_EPT; ++e) {
        if (base + e >= M) break;
        const unsigned int d = (k[e] >> shift) & 255u;
        const unsigned int r = cnt[d * SORT_STRIDE + t];
        cnt[d * SORT_STRIDE + t] = (unsigned short)(r + 1);
        const unsigned int dst = hist[(long long)d * ntiles + blockIdx.x] + r;
        key_out[dst] = k[e];
        idx_out[dst] = ix[e];
    }
}

// the five per-point arrays in sorted order
template <typename T>
__global__ void __launch_bounds__(256) gather_obs_kernel(const unsigned int* __restrict__ perm, long long M,
                                                         const T* __restrict__ u, const T* __restrict__ v,
                                                         const T* __restrict__ re, const T* __restrict__ im,
                                                         const T* __restrict__ w, T* __restrict__ su, T* __restrict__ sv,
                                                         T* __restrict__ sre, T* __restrict__ sim, T* __restrict__ sw) {
    for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k < M; k += (long long)gridDim.x * blockDim.x) {
        const unsigned int s = perm[k];
        su[k] = u[s]; sv[k] = v[s]; sre[k] = re[s]; sim[k] = im[s]; sw[k] = w[s];
    }
}

}  // namespace galb
