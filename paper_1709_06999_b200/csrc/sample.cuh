// sample.cuh — fused rotate (S5) + bilinear gather (S6) + phase ramp (S7) + chi-square (S8).
//
// One kernel does the whole per-point part of the paper's listing so that for
// chi2* the visibilities never go to memory ("the purpose of the Chi2* function is
// to avoid transferring the sampled visibilities back").  The index arithmetic follows the listing
// operation by operation, each one individually rounded in double (no FMA contraction), so the
// cell an (u, v) point falls in and its weights are decided exactly as a plain IEEE evaluation of
// the listing decides them — in _f32 as well (reading A14).
// The spectrum is the u-major array written by fft.cuh: spec[ku][kvs].
//
// Data movement (sm_100a):
//   * the per-point arrays u, v, re_obs, im_obs, w are streamed by the TMA engine: one elected
//     thread issues `cp.async.bulk` copies of whole tiles (256*U points of each array) into a ring
//     of shared-memory stages, completion signalled on an mbarrier.  The loads cost no registers,
//     no LSU wavefronts and are always STAGES-1 tiles ahead of the arithmetic;
//   * the four spectrum nodes of a point are gathered by lane pairs through the L1 (see below);
//     that gather — one L1 wavefront per 128-byte line touched — is what bounds the kernel once
//     the streams are off the LSU, so everything else is arranged to overlap with it.
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
    double cos_PA, sin_PA;
    double dRA_turns, dDec_turns;  // rotated offsets in turns: theta / 2 pi = u' dRA_turns + v' dDec_turns
    int has_phase;         // 0 when both rotated offsets are 0 (theta == 0 exactly)
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

// The listing's index arithmetic for one point (Eq. 11-12, 676-683), shared by the
// sampler and the uv-extent kernel so both take the same integer decisions.
struct PointIndex {
    double urot, vrot, uidx, vidx;
    bool uneg;
};
template <typename P>
__device__ __forceinline__ PointIndex point_index(const P& p, double u, double v, double fH) {
    PointIndex q;
    q.urot = __dsub_rn(__dmul_rn(u, p.cos_PA), __dmul_rn(v, p.sin_PA));
    q.vrot = __dadd_rn(__dmul_rn(u, p.sin_PA), __dmul_rn(v, p.cos_PA));
    q.uidx = div_by(fabs(q.urot), p.du, p.rdu, p.du_exact_div);
    q.uneg = q.urot < 0.0;
    const double vq = div_by(q.vrot, p.du, p.rdu, p.du_exact_div);
    q.vidx = q.uneg ? __dsub_rn(fH, vq) : __dadd_rn(fH, vq);
    return q;
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

// ------------------------------------------------------------------------------------------
// uv extent: which part of the half plane can the point set reach?
// ext[0] = largest column ku any interpolation cell touches, ext[1] / ext[2] = smallest / largest
// shifted row kvs; a point whose cell leaves the grid (reading A6: the wrap can reach anything)
// sets the full extent.  Integer max/min only, so the result does not depend on the order.
// The FFT passes skip what lies outside (fft.cuh), which changes no result.
// ------------------------------------------------------------------------------------------
struct ExtentParams {
    int N;
    long long total;       // C * M
    double du, rdu;
    int du_exact_div;
    double cos_PA, sin_PA;
    int* ext;              // [3], initialised to {0, N-1, 0} by the host
};

template <typename T>
__global__ void __launch_bounds__(256) uv_extent_kernel(const ExtentParams p, const T* __restrict__ u,
                                                        const T* __restrict__ v) {
    const int N = p.N, H = N >> 1;
    const double fH = (double)H, fN1 = (double)(N - 1);
    int cmax = 0, rmin = N - 1, rmax = 0;
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k < p.total; k += stride) {
        const PointIndex q = point_index(p, (double)__ldcs(u + k), (double)__ldcs(v + k), fH);
        const bool inside = q.uidx <= fH - 1.0 && q.vidx >= 0.0 && q.vidx < fN1;
        if (inside) {
            const int ix = (int)q.uidx, iy = (int)q.vidx;      // both >= 0: truncation == floor
            cmax = max(cmax, ix + 1);
            rmin = min(rmin, iy);
            rmax = max(rmax, iy + 1);
        } else {
            cmax = H; rmin = 0; rmax = N - 1;
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        cmax = max(cmax, __shfl_xor_sync(0xffffffffu, cmax, o));
        rmin = min(rmin, __shfl_xor_sync(0xffffffffu, rmin, o));
        rmax = max(rmax, __shfl_xor_sync(0xffffffffu, rmax, o));
    }
    if ((threadIdx.x & 31) == 0) {
        atomicMax(p.ext + 0, cmax);
        atomicMin(p.ext + 1, rmin);
        atomicMax(p.ext + 2, rmax);
    }
}

// ------------------------------------------------------------------------------------------
// mbarrier + TMA bulk-copy wrappers (PTX, sm_90+/sm_100a).
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t mb, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(mb), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint32_t mb, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(mb), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t mb, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(mb), "r"(parity) : "memory");
}
__device__ __forceinline__ uint64_t l2_policy_evict_first() {
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
// global -> shared bulk copy (TMA, 1-D): 16-byte aligned addresses, size a multiple of 16 bytes.
__device__ __forceinline__ void tma_load_1d(uint32_t dst, const void* src, uint32_t bytes, uint32_t mb, uint64_t pol) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
        ::"r"(dst), "l"(src), "r"(bytes), "r"(mb), "l"(pol) : "memory");
}

// Points per thread and tile (U), stages of the shared-memory ring, resident CTAs per SM the register
// budget is set for.
#ifndef GAL_SAMPLE_U
#define GAL_SAMPLE_U 2
#endif
#ifndef GAL_SAMPLE_STAGES
#define GAL_SAMPLE_STAGES 3
#endif
#ifndef GAL_SAMPLE_MINB
#define GAL_SAMPLE_MINB 3
#endif

template <typename T, bool DO_CHI2> struct SampleGeom {
    static constexpr int U = GAL_SAMPLE_U;
    static constexpr int NT = 256;
    static constexpr int TILE = NT * U;
    static constexpr int NARR = DO_CHI2 ? 5 : 2;
    static constexpr int S = GAL_SAMPLE_STAGES;
    static constexpr uint32_t ARR_BYTES = TILE * sizeof(T);
    static constexpr uint32_t STAGE_BYTES = NARR * ARR_BYTES;
    static constexpr size_t SMEM = (size_t)S * STAGE_BYTES + 8 * S;
};

// Gather by lane pairs.  The four nodes of a cell are two 32-byte runs (kvs, kvs+1 at ku and at ku+1) in
// the u-major spectrum.  The L1 serves about one 128-byte line per clock, whatever the width of the access
// (measured: 0.8-1.0 clk per line touched by an LDG), and a point needs 2.25 lines, so a warp-wide 16-byte
// load of 32 unrelated nodes would spend 32 clocks for 32 nodes.  Lanes 2i and 2i+1 therefore fetch each
// other's cells together: in every load instruction the even lane reads node kvs and the odd lane node
// kvs+1 of the SAME cell — one line per lane pair.  Each lane then forms the u-direction interpolation of
// its row for both cells, one shuffle hands the row the partner needs across, and the owner finishes its
// own point.
template <typename T, bool WRITE_VIS, bool DO_CHI2, bool TMA>
__global__ void __launch_bounds__(256, GAL_SAMPLE_MINB) sample_kernel(const SampleParams<T> p) {
    using G = SampleGeom<T, DO_CHI2>;
    constexpr int U = G::U, TILE = G::TILE, S = G::S;
    extern __shared__ __align__(128) unsigned char sample_smem[];
    const int tid = threadIdx.x;
    const int c = blockIdx.y;
    const int N = p.N, H = N >> 1;
    const long long M = p.M;
    const cx<T>* __restrict__ spec = p.spec + (long long)c * (H + 1) * N;
    const T* __restrict__ gsrc[5] = {p.u + c * M, p.v + c * M, DO_CHI2 ? p.re_obs + c * M : nullptr,
                                     DO_CHI2 ? p.im_obs + c * M : nullptr, DO_CHI2 ? p.w + c * M : nullptr};
    const double fH = (double)H, fN1 = (double)(N - 1);
    const int odd = tid & 1;
    const long long ntiles = (M + TILE - 1) / TILE, nfull = M / TILE;

    // ---- TMA producer: thread 0 keeps S-1 tiles in flight ----
    const uint32_t bar0 = smem_u32(sample_smem + (size_t)S * G::STAGE_BYTES);
    uint64_t pol = 0;
    auto issue = [&](long long tile, int s) {
        if (tile >= nfull) return;                       // the ragged last tile is read with plain loads
        const uint32_t mb = bar0 + 8 * s;
        const uint32_t dst = smem_u32(sample_smem + (size_t)s * G::STAGE_BYTES);
        mbar_expect_tx(mb, G::STAGE_BYTES);
#pragma unroll
        for (int a = 0; a < G::NARR; ++a) tma_load_1d(dst + a * G::ARR_BYTES, gsrc[a] + tile * TILE, G::ARR_BYTES, mb, pol);
    };
    if (TMA) {
        if (tid == 0) {
            for (int s = 0; s < S; ++s) mbar_init(bar0 + 8 * s, 1);
            mbar_fence_init();
            pol = l2_policy_evict_first();
            for (int s = 0; s < S - 1; ++s) issue(blockIdx.x + (long long)s * gridDim.x, s);
        }
    }

    double acc = 0.0;
    unsigned int oob = 0;
    int it = 0;
    for (long long tile = blockIdx.x; tile < ntiles; tile += gridDim.x, ++it) {
        const int s = it % S;
        const bool staged = TMA && tile < nfull;
        if (TMA) {
            __syncthreads();                             // stage (it-1) % S has been consumed by everyone
            if (tid == 0) issue(tile + (long long)(S - 1) * gridDim.x, (it + S - 1) % S);
            if (staged) mbar_wait(bar0 + 8 * s, (uint32_t)(it / S) & 1u);
        }
        const T* st = reinterpret_cast<const T*>(sample_smem + (size_t)s * G::STAGE_BYTES);
        const long long k0 = tile * TILE + tid;

        double tx[U], ty[U], ro[U], io[U], wt[U];
        PointIndex q[U];
        bool inside[U];
        cx<T> ga0[U], ga1[U], gb0[U], gb1[U];   // even lane's cell (a) / odd lane's cell (b); column ku+0 / ku+1
#pragma unroll
        for (int j = 0; j < U; ++j) {
            double pu = 0.0, pv = 0.0;                   // dead slots: index (0, N/2), weight 0
            ro[j] = io[j] = wt[j] = 0.0;
            if (staged) {
                pu = (double)st[0 * TILE + j * 256 + tid];
                pv = (double)st[1 * TILE + j * 256 + tid];
                if (DO_CHI2) {
                    ro[j] = (double)st[2 * TILE + j * 256 + tid];
                    io[j] = (double)st[3 * TILE + j * 256 + tid];
                    wt[j] = (double)st[4 * TILE + j * 256 + tid];
                }
            } else if (k0 + j * 256 < M) {
                const long long k = k0 + j * 256;
                pu = (double)__ldcs(gsrc[0] + k);
                pv = (double)__ldcs(gsrc[1] + k);
                if (DO_CHI2) {
                    ro[j] = (double)__ldcs(gsrc[2] + k);
                    io[j] = (double)__ldcs(gsrc[3] + k);
                    wt[j] = (double)__ldcs(gsrc[4] + k);
                }
            }
            q[j] = point_index(p, pu, pv, fH);
            // bilinear interpolation
            const double fx0 = floor(q[j].uidx), fy0 = floor(q[j].vidx);
            tx[j] = __dsub_rn(q[j].uidx, fx0);
            ty[j] = __dsub_rn(q[j].vidx, fy0);
            inside[j] = q[j].uidx <= fH - 1.0 && q[j].vidx >= 0.0 && q[j].vidx < fN1;   // cell fully inside the grid
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
            // this lane's row (kvs + odd) of both cells, interpolated along u: g0 + t (g1 - g0)
            const double ra_re = fma(txa, (double)ga1[j].x - (double)ga0[j].x, (double)ga0[j].x);
            const double ra_im = fma(txa, (double)ga1[j].y - (double)ga0[j].y, (double)ga0[j].y);
            const double rb_re = fma(txb, (double)gb1[j].x - (double)gb0[j].x, (double)gb0[j].x);
            const double rb_im = fma(txb, (double)gb1[j].y - (double)gb0[j].y, (double)gb0[j].y);
            // the even lane needs row kvs+1 of cell a, the odd lane row kvs of cell b
            const double o_re = __shfl_xor_sync(0xffffffffu, odd ? ra_re : rb_re, 1);
            const double o_im = __shfl_xor_sync(0xffffffffu, odd ? ra_im : rb_im, 1);
            const double lo_re = odd ? o_re : ra_re, hi_re = odd ? rb_re : o_re;
            const double lo_im = odd ? o_im : ra_im, hi_im = odd ? rb_im : o_im;
            double ReInt = fma(ty[j], hi_re - lo_re, lo_re);
            double ImInt = fma(ty[j], hi_im - lo_im, lo_im);
            if (!inside[j]) {           // rare: the cell leaves the half-plane grid (reading A6); dead slots never get here
                const double uidx = q[j].uidx, vidx = q[j].vidx;
                const long long ix = (long long)floor(uidx), iy = (long long)floor(vidx);
                if (uidx > fH || vidx < 0.0 || vidx > fN1) ++oob;
                const cx<T> g00 = node_any<T>(spec, N, iy, ix), g01 = node_any<T>(spec, N, iy, ix + 1);
                const cx<T> g10 = node_any<T>(spec, N, iy + 1, ix), g11 = node_any<T>(spec, N, iy + 1, ix + 1);
                const double ax = 1.0 - tx[j], ay = 1.0 - ty[j];
                ReInt = ay * (ax * (double)g00.x + tx[j] * (double)g01.x) + ty[j] * (ax * (double)g10.x + tx[j] * (double)g11.x);
                ImInt = ay * (ax * (double)g00.y + tx[j] * (double)g01.y) + ty[j] * (ax * (double)g10.y + tx[j] * (double)g11.y);
            }
            if (q[j].uneg) ImInt = -ImInt;
            double vr = ReInt, vi = ImInt;
            if (p.has_phase) {                                  // PAPER.md:712-713, theta in turns: exact range reduction
                const double turns = fma(q[j].urot, p.dRA_turns, q[j].vrot * p.dDec_turns);
                double sn, co;
                sincospi(2.0 * turns, &sn, &co);
                vr = ReInt * co - ImInt * sn;
                vi = ReInt * sn + ImInt * co;
            }
            if (WRITE_VIS) {
                const long long k = k0 + j * 256;
                if (k < M) __stcs(reinterpret_cast<cx<T>*>(p.vis) + c * M + k, mk<T>((T)vr, (T)vi));
            }
            if (DO_CHI2) {                                      // PAPER.md:718 (Eq. 10); w = 0 for dead slots
                const double dr = vr - ro[j];
                const double di = vi - io[j];
                acc = fma(fma(dr, dr, di * di), wt[j], acc);
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
