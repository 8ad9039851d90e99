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
// periodicity and Hermitian symmetry of the DFT of a real image (reading A6).  Rare path (points
// beyond the half-plane grid), kept out of line.
template <typename T>
__device__ __noinline__ cx<T> node_any(const cx<T>* __restrict__ spec, int N, long long row, long long col) {
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

// Points per thread and loop trip (U), and resident CTAs per SM the register budget is set for.
// Per trip: the streamed inputs of the NEXT trip are requested first (register double buffer), then
// the 4U spectrum nodes of this trip, then the arithmetic — so the DRAM latency of the per-point
// arrays is off the critical path and only the (mostly L2-resident) gather latency is exposed.
#ifndef GAL_SAMPLE_U
#define GAL_SAMPLE_U 2
#endif
#ifndef GAL_SAMPLE_MINB
#define GAL_SAMPLE_MINB 2
#endif

template <typename T, bool DO_CHI2> struct PointIn {
    double u, v, ro, io, w;
};

template <typename T, bool DO_CHI2>
__device__ __forceinline__ void load_point(PointIn<T, DO_CHI2>& q, const T* __restrict__ u, const T* __restrict__ v,
                                           const T* __restrict__ re, const T* __restrict__ im,
                                           const T* __restrict__ w, long long k, long long M) {
    q.u = q.v = q.ro = q.io = q.w = 0.0;            // dead slots: index (0, N/2), weight 0
    if (k < M) {
        q.u = (double)__ldcs(u + k);
        q.v = (double)__ldcs(v + k);
        if (DO_CHI2) {
            q.ro = (double)__ldcs(re + k);
            q.io = (double)__ldcs(im + k);
            q.w = (double)__ldcs(w + k);
        }
    }
}

// Gather by lane pairs.  The four nodes of a cell are two 32-byte runs (kvs, kvs+1 at ku and at ku+1) in
// the u-major spectrum.  A warp-wide 16-byte load of 32 unrelated addresses costs the L1 32 tag look-ups,
// and with four of them per point that look-up rate (one line per clock and SM) is what bounds the kernel,
// not HBM.  So lanes 2i and 2i+1 fetch each other's cells together: in every load instruction the even
// lane reads node kvs and the odd lane node kvs+1 of the SAME cell — one line per lane pair, 16-18 lines
// per instruction instead of 32.  Each lane then forms the u-direction interpolation of its row for both
// cells, one shuffle hands the row the partner needs across, and the owner finishes its own point.
template <typename T, bool WRITE_VIS, bool DO_CHI2>
__global__ void __launch_bounds__(256, GAL_SAMPLE_MINB) sample_kernel(const SampleParams<T> p) {
    constexpr int U = GAL_SAMPLE_U;
    const int c = blockIdx.y;
    const int N = p.N, H = N >> 1;
    const long long M = p.M;
    const cx<T>* __restrict__ spec = p.spec + (long long)c * (H + 1) * N;
    const T* __restrict__ u = p.u + c * M;
    const T* __restrict__ v = p.v + c * M;
    const T* __restrict__ re_obs = DO_CHI2 ? p.re_obs + c * M : nullptr;
    const T* __restrict__ im_obs = DO_CHI2 ? p.im_obs + c * M : nullptr;
    const T* __restrict__ wgt = DO_CHI2 ? p.w + c * M : nullptr;
    const double fH = (double)H, fN1 = (double)(N - 1);
    const int odd = threadIdx.x & 1;

    double acc = 0.0;
    unsigned int oob = 0;
    const long long stride = (long long)gridDim.x * blockDim.x * U;
    long long k0 = (long long)blockIdx.x * blockDim.x * U + threadIdx.x;
    long long kw = k0 - (threadIdx.x & 31);                 // warp-uniform: every lane takes every trip
    PointIn<T, DO_CHI2> nxt[U];
#pragma unroll
    for (int j = 0; j < U; ++j) load_point<T, DO_CHI2>(nxt[j], u, v, re_obs, im_obs, wgt, k0 + (long long)j * blockDim.x, M);
    for (; kw < M; kw += stride, k0 += stride) {
        PointIn<T, DO_CHI2> cur[U];
#pragma unroll
        for (int j = 0; j < U; ++j) cur[j] = nxt[j];
#pragma unroll
        for (int j = 0; j < U; ++j)
            load_point<T, DO_CHI2>(nxt[j], u, v, re_obs, im_obs, wgt, k0 + stride + (long long)j * blockDim.x, M);

        double urot[U], vrot[U], tx[U], ty[U], uidx[U], vidx[U];
        bool uneg[U], inside[U];
        cx<T> ga0[U], ga1[U], gb0[U], gb1[U];   // even lane's cell (a) / odd lane's cell (b); column ku+0 / ku+1
#pragma unroll
        for (int j = 0; j < U; ++j) {
            // PAPER.md:667-668 (Eq. 11-12)
            urot[j] = __dsub_rn(__dmul_rn(cur[j].u, p.cos_PA), __dmul_rn(cur[j].v, p.sin_PA));
            vrot[j] = __dadd_rn(__dmul_rn(cur[j].u, p.sin_PA), __dmul_rn(cur[j].v, p.cos_PA));
            // PAPER.md:676-683
            uidx[j] = div_by(fabs(urot[j]), p.du, p.rdu, p.du_exact_div);
            uneg[j] = urot[j] < 0.0;
            const double vq = div_by(vrot[j], p.du, p.rdu, p.du_exact_div);
            vidx[j] = uneg[j] ? __dsub_rn(fH, vq) : __dadd_rn(fH, vq);
            // bilinear interpolation
            const double fx0 = floor(uidx[j]), fy0 = floor(vidx[j]);
            tx[j] = __dsub_rn(uidx[j], fx0);
            ty[j] = __dsub_rn(vidx[j], fy0);
            inside[j] = uidx[j] <= fH - 1.0 && vidx[j] >= 0.0 && vidx[j] < fN1;     // cell fully inside the grid
            const int off = inside[j] ? (int)fx0 * N + (int)fy0 : 0;
            const int off_partner = __shfl_xor_sync(0xffffffffu, off, 1);
            const cx<T>* pa = spec + ((odd ? off_partner : off) + odd);
            const cx<T>* pb = spec + ((odd ? off : off_partner) + odd);
            ga0[j] = __ldg(pa);
            ga1[j] = __ldg(pa + N);
            gb0[j] = __ldg(pb);
            gb1[j] = __ldg(pb + N);
        }
#pragma unroll
        for (int j = 0; j < U; ++j) {
            const double tx_partner = __shfl_xor_sync(0xffffffffu, tx[j], 1);
            const double txa = odd ? tx_partner : tx[j], txb = odd ? tx[j] : tx_partner;
            const double axa = 1.0 - txa, axb = 1.0 - txb;
            // this lane's row (kvs + odd) of both cells, interpolated along u
            const double ra_re = axa * (double)ga0[j].x + txa * (double)ga1[j].x;
            const double ra_im = axa * (double)ga0[j].y + txa * (double)ga1[j].y;
            const double rb_re = axb * (double)gb0[j].x + txb * (double)gb1[j].x;
            const double rb_im = axb * (double)gb0[j].y + txb * (double)gb1[j].y;
            // the even lane needs row kvs+1 of cell a, the odd lane row kvs of cell b
            const double o_re = __shfl_xor_sync(0xffffffffu, odd ? ra_re : rb_re, 1);
            const double o_im = __shfl_xor_sync(0xffffffffu, odd ? ra_im : rb_im, 1);
            const double ay = 1.0 - ty[j];
            double ReInt = odd ? ay * o_re + ty[j] * rb_re : ay * ra_re + ty[j] * o_re;
            double ImInt = odd ? ay * o_im + ty[j] * rb_im : ay * ra_im + ty[j] * o_im;
            if (!inside[j]) {           // rare: the cell leaves the half-plane grid (reading A6); dead slots never get here
                const long long ix = (long long)floor(uidx[j]), iy = (long long)floor(vidx[j]);
                if (uidx[j] > fH || vidx[j] < 0.0 || vidx[j] > fN1) ++oob;
                const cx<T> g00 = node_any<T>(spec, N, iy, ix), g01 = node_any<T>(spec, N, iy, ix + 1);
                const cx<T> g10 = node_any<T>(spec, N, iy + 1, ix), g11 = node_any<T>(spec, N, iy + 1, ix + 1);
                const double ax = 1.0 - tx[j];
                ReInt = ay * (ax * (double)g00.x + tx[j] * (double)g01.x) + ty[j] * (ax * (double)g10.x + tx[j] * (double)g11.x);
                ImInt = ay * (ax * (double)g00.y + tx[j] * (double)g01.y) + ty[j] * (ax * (double)g10.y + tx[j] * (double)g11.y);
            }
            if (uneg[j]) ImInt = -ImInt;
            double vr = ReInt, vi = ImInt;
            if (p.has_phase) {
                const double theta = __dadd_rn(__dmul_rn(urot[j], p.dRArot), __dmul_rn(vrot[j], p.dDecrot));
                double sn, co;
                sincos(theta, &sn, &co);
                vr = ReInt * co - ImInt * sn;
                vi = ReInt * sn + ImInt * co;
            }
            if (WRITE_VIS) {
                const long long k = k0 + (long long)j * blockDim.x;
                if (k < M) __stcs(reinterpret_cast<cx<T>*>(p.vis) + c * M + k, mk<T>((T)vr, (T)vi));
            }
            if (DO_CHI2) {                                      // PAPER.md:718 (Eq. 10); w = 0 for dead slots
                const double dr = vr - cur[j].ro;
                const double di = vi - cur[j].io;
                acc += (dr * dr + di * di) * cur[j].w;
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
