// sample.cuh — fused rotate (S5) + bilinear gather (S6) + phase ramp (S7) + chi-square (S8).
//
// One kernel does the whole per-point part of the paper's listing so that for
// chi2* the visibilities never go to memory ("the purpose of the Chi2* function is
// to avoid transferring the sampled visibilities back").  The index and phase arithmetic follows
// the listing operation by operation, each one individually rounded in double (no FMA
// contraction), so the cell an (u, v) point falls in and its weights are decided exactly as a
// plain IEEE evaluation of the listing decides them — in _f32 as well (reading A14).
// The spectrum is the u-major array written by fft.cuh: spec[ku][kvs].
#pragma once
#include "fft.cuh"

namespace galb {

template <typename T> struct SampleParams {
    const cx<T>* spec;     // [C][N/2+1][N]
    int N;
    long long M;           // points per channel
    const T* u; const T* v;                       // [C][M]
    const T* re_obs; const T* im_obs; const T* w; // [C][M] (chi2 only)
    T* vis;                                       // [C][2M] (sample only)
    double du, rdu;        // du = 1/(N dxy); rdu = RN(1/du) for the exact-division shortcut
    int du_exact_div;      // 1: use a true division (rdu not usable)
    double cos_PA, sin_PA, dRArot, dDecrot;
    int has_phase;         // 0 when dRArot == dDecrot == 0 (theta == 0 exactly)
    double* partials;      // [C][gridDim.x]
    unsigned int* tickets; // [C + 1]
    double* chi2_per_channel; // [C] or null
    double* chi2_total;       // [1] or null
    unsigned long long* oob;  // [1]
};

// Correctly rounded a / b from r = RN(1/b) (Markstein): q0 = RN(a r); rem = a - q0 b (exact in an
// FMA); q = RN(q0 + rem r).  Bit-identical to __ddiv_rn for the operand ranges met here (finite,
// normal, b without an all-ones significand — the host checks b and otherwise asks for a true
// division).
__device__ __forceinline__ double div_by(double a, double b, double r, int exact) {
    if (exact) return __ddiv_rn(a, b);
    const double q0 = __dmul_rn(a, r);
    const double rem = __fma_rn(-q0, b, a);
    return __fma_rn(rem, r, q0);
}

// Node (row = shifted v index, col = u index) of the spectrum extended to all integers by the
// periodicity and Hermitian symmetry of the DFT of a real image (reading A6).
template <typename T>
__device__ __forceinline__ cx<T> node_any(const cx<T>* __restrict__ spec, int N, long long row, long long col) {
    const int H = N >> 1;
    long long kv = row - H;
    long long cu = col & (long long)(N - 1);          // N is a power of two: floor-mod
    if (cu <= H) {
        const long long r = ((kv & (N - 1)) + H) & (N - 1);
        return __ldg(spec + cu * N + r);
    }
    const long long r = (((-kv) & (N - 1)) + H) & (N - 1);
    cx<T> g = __ldg(spec + (N - cu) * N + r);
    g.y = -g.y;
    return g;
}

// Points per thread and loop trip.  All streamed inputs of the U points are requested first, then the
// 4U spectrum nodes, then the arithmetic: three dependent memory latencies per trip instead of per point.
constexpr int SAMPLE_U = 2;

template <typename T, bool WRITE_VIS, bool DO_CHI2>
__global__ void __launch_bounds__(256) sample_kernel(const SampleParams<T> p) {
    constexpr int U = SAMPLE_U;
    const int c = blockIdx.y;
    const int N = p.N, H = N >> 1;
    const long long M = p.M;
    const cx<T>* __restrict__ spec = p.spec + (long long)c * (H + 1) * N;
    const T* __restrict__ u = p.u + c * M;
    const T* __restrict__ v = p.v + c * M;
    const T* __restrict__ re_obs = DO_CHI2 ? p.re_obs + c * M : nullptr;
    const T* __restrict__ im_obs = DO_CHI2 ? p.im_obs + c * M : nullptr;
    const T* __restrict__ wgt = DO_CHI2 ? p.w + c * M : nullptr;
    const double fH = (double)H;

    double acc = 0.0;
    unsigned int oob = 0;
    const long long stride = (long long)gridDim.x * blockDim.x * U;
    for (long long k0 = (long long)blockIdx.x * blockDim.x * U + threadIdx.x; k0 < M; k0 += stride) {
        double uk[U], vk[U], ro[U], io[U], wk[U];
        bool live[U];
#pragma unroll
        for (int j = 0; j < U; ++j) {
            const long long k = k0 + (long long)j * blockDim.x;
            live[j] = k < M;
            uk[j] = vk[j] = ro[j] = io[j] = wk[j] = 0.0;
            if (live[j]) {
                uk[j] = (double)__ldcs(u + k);
                vk[j] = (double)__ldcs(v + k);
                if (DO_CHI2) {
                    ro[j] = (double)__ldcs(re_obs + k);
                    io[j] = (double)__ldcs(im_obs + k);
                    wk[j] = (double)__ldcs(wgt + k);
                }
            }
        }
        double urot[U], vrot[U], tx[U], ty[U];
        bool uneg[U];
        cx<T> g00[U], g01[U], g10[U], g11[U];   // g{row offset}{col offset}
#pragma unroll
        for (int j = 0; j < U; ++j) {
            // PAPER.md:667-668 (Eq. 11-12)
            urot[j] = __dsub_rn(__dmul_rn(uk[j], p.cos_PA), __dmul_rn(vk[j], p.sin_PA));
            vrot[j] = __dadd_rn(__dmul_rn(uk[j], p.sin_PA), __dmul_rn(vk[j], p.cos_PA));
            // PAPER.md:676-683
            const double urot_idx = div_by(fabs(urot[j]), p.du, p.rdu, p.du_exact_div);
            uneg[j] = urot[j] < 0.0;
            const double vq = div_by(vrot[j], p.du, p.rdu, p.du_exact_div);
            const double vrot_idx = uneg[j] ? __dsub_rn(fH, vq) : __dadd_rn(fH, vq);
            if (live[j] && (urot_idx > fH || vrot_idx < 0.0 || vrot_idx > (double)(N - 1))) ++oob;
            // bilinear interpolation
            const double fx0 = floor(urot_idx), fy0 = floor(vrot_idx);
            const long long ix = (long long)fx0, iy = (long long)fy0;
            tx[j] = __dsub_rn(urot_idx, fx0);
            ty[j] = __dsub_rn(vrot_idx, fy0);
            if (ix + 1 <= H && iy >= 0 && iy + 1 <= N - 1) {
                const cx<T>* b0 = spec + ix * N + iy;
                g00[j] = __ldg(b0);
                g10[j] = __ldg(b0 + 1);
                g01[j] = __ldg(b0 + N);
                g11[j] = __ldg(b0 + N + 1);
            } else {
                g00[j] = node_any<T>(spec, N, iy, ix);
                g01[j] = node_any<T>(spec, N, iy, ix + 1);
                g10[j] = node_any<T>(spec, N, iy + 1, ix);
                g11[j] = node_any<T>(spec, N, iy + 1, ix + 1);
            }
        }
#pragma unroll
        for (int j = 0; j < U; ++j) {
            const double ax = 1.0 - tx[j], ay = 1.0 - ty[j];
            double ReInt = ay * (ax * (double)g00[j].x + tx[j] * (double)g01[j].x) +
                           ty[j] * (ax * (double)g10[j].x + tx[j] * (double)g11[j].x);
            double ImInt = ay * (ax * (double)g00[j].y + tx[j] * (double)g01[j].y) +
                           ty[j] * (ax * (double)g10[j].y + tx[j] * (double)g11[j].y);
            if (uneg[j]) ImInt = -ImInt;
            double vr = ReInt, vi = ImInt;
            if (p.has_phase) {
                const double theta = __dadd_rn(__dmul_rn(urot[j], p.dRArot), __dmul_rn(vrot[j], p.dDecrot));
                double sn, co;
                sincos(theta, &sn, &co);
                vr = ReInt * co - ImInt * sn;
                vi = ReInt * sn + ImInt * co;
            }
            if (WRITE_VIS && live[j]) {
                cx<T>* out = reinterpret_cast<cx<T>*>(p.vis) + c * M + k0 + (long long)j * blockDim.x;
                __stcs(out, mk<T>((T)vr, (T)vi));
            }
            if (DO_CHI2) {                                      // PAPER.md:718 (Eq. 10); wk = 0 for dead slots
                const double dr = vr - ro[j];
                const double di = vi - io[j];
                acc += (dr * dr + di * di) * wk[j];
            }
        }
    }

    // ---- deterministic reduction: warp shuffle -> block -> per-block partial -> last block ----
    __shared__ double wsum[8];
    __shared__ unsigned int woob[8];
    __shared__ bool is_last;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        acc += __shfl_down_sync(0xffffffffu, acc, o);
        oob += __shfl_down_sync(0xffffffffu, oob, o);
    }
    if (lane == 0) { wsum[wid] = acc; woob[wid] = oob; }
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = 0.0;
        unsigned int ob = 0;
        for (int i = 0; i < (int)(blockDim.x >> 5); ++i) { s += wsum[i]; ob += woob[i]; }
        if (ob) atomicAdd(p.oob, (unsigned long long)ob);
        if (DO_CHI2) {
            p.partials[(long long)c * gridDim.x + blockIdx.x] = s;
            __threadfence();
            const unsigned int tk = atomicAdd(&p.tickets[c], 1u);
            is_last = (tk == gridDim.x - 1);
        }
    }
    if (!DO_CHI2) return;
    __syncthreads();
    if (!is_last) return;
    // last block of this channel: sum the partials in index order with a fixed tree
    __threadfence();
    double s = 0.0;
    const volatile double* part = p.partials + (long long)c * gridDim.x;
    for (int i = threadIdx.x; i < (int)gridDim.x; i += blockDim.x) s += part[i];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_down_sync(0xffffffffu, s, o);
    __syncthreads();
    if (lane == 0) wsum[wid] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        double tot = 0.0;
        for (int i = 0; i < (int)(blockDim.x >> 5); ++i) tot += wsum[i];
        if (p.chi2_per_channel) p.chi2_per_channel[c] = tot;
        p.tickets[c] = 0;                                       // re-arm for the next call
        if (p.chi2_total) {
            __threadfence();
            const unsigned int tk = atomicAdd(&p.tickets[gridDim.y], 1u);
            if (tk == gridDim.y - 1) {                          // last channel to finish: total in channel order
                __threadfence();
                double t = 0.0;
                if (p.chi2_per_channel) {
                    const volatile double* pc = p.chi2_per_channel;
                    for (int i = 0; i < (int)gridDim.y; ++i) t += pc[i];
                } else {
                    t = tot;                                    // single channel
                }
                *p.chi2_total = t;
                p.tickets[gridDim.y] = 0;
            }
        }
    }
}

}  // namespace galb
