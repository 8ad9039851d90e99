// sample.cuh — fused rotate (S5) + bilinear gather (S6) + phase ramp (S7) + chi-square (S8).
//
// One kernel does the whole per-point part of the paper's listing so that for
// chi2* the visibilities never go to memory ("the purpose of the Chi2* function is
// to avoid transferring the sampled visibilities back").  The index arithmetic follows the listing
// operation by operation, each one individually rounded in double (no FMA contraction), so the
// cell an (u, v) point falls in and its weights are decided exactly as a plain IEEE evaluation of
// the listing decides them — in _f32 as well (reading A14).
// The spectrum is the u-major array of column pairs written by fft.cuh: pair[ku][kvs] = {F[ku][kvs], F[ku+1][kvs]}.
//
// Data movement (sm_100a):
//   * the per-point arrays u, v, re_obs, im_obs, w are streamed by the TMA engine: a producer warp
//     issues `cp.async.bulk` copies of whole tiles (256*U points of each array) into a ring of
//     shared-memory stages, full/empty mbarriers hand the stages back and forth.  The loads cost the
//     consumer warps no registers, no instructions and no L1 tag look-ups, and run up to STAGES
//     tiles ahead of the arithmetic;
//   * the four spectrum nodes of a point are gathered by lane pairs through the L1 (see below);
//     that gather is bounded by the L2 -> SM path and by the L1's one line per clock, so it is
//     shaped to move the fewest sectors and lines, and everything else overlaps with it.
#pragma once
#include <type_traits>

#include "common.cuh"

namespace galb {

template <typename T> struct SampleParams {
    const NodePair<T>* spec;   // [C][N/2+1][N] column pairs (fft.cuh)
    int N;
    long long M;           // points per channel
    const T* u; const T* v;                       // [C][M]
    const T* re_obs; const T* im_obs; const T* w; // [C][M] (chi2 only)
    T* vis;                                       // [C][2M] (sample only)
    IndexScalars ix;
    double dRA_turns, dDec_turns;  // rotated offsets in turns: theta / 2 pi = u' dRA_turns + v' dDec_turns
    int has_phase;         // 0 when both rotated offsets are 0 (theta == 0 exactly)
    double amp;            // factor on the visibilities (1 except for multi-source composition)
    int accumulate;        // sample*: add to what vis already holds (sources after the first) instead of storing
    double* partials;      // [C][gridDim.x]
    unsigned int* tickets; // [C + 1]
    double* chi2_per_channel; // [C] or null
    double* chi2_total;       // [1] or null
    unsigned long long* oob;  // [1]: this call's out-of-grid counter
    unsigned int* done;       // [1]: CTAs of this launch that have finished
    unsigned long long* next_state;  // the copy of the per-call state the NEXT call will use (32 B)
    const int* ext;           // the extent the transform was pruned to: whole plane = single-copy layout (fft.cuh)
    const int* ext_check;     // extent of a bound uv set to verify every point against, or null
    unsigned long long* viol; // [1]: points whose cell lies outside ext_check
    int direct;               // 1: every thread gathers its own cell (uv-sorted points of a bound observation set)
    int shared_spec;          // 1: every channel (blockIdx.y) samples the ONE spectrum at spec (K observation sets against one image)
    int rearm;                // 1: the last CTA of this launch re-arms next_state (every launch but the non-final chunks of a long multi-source list)
    unsigned int* viol_flag;  // mapped host memory: set when viol becomes non-zero (sticky, read by the next call)
    unsigned int* ext_hint;   // mapped host memory or null: 1 = this call's extent was the whole plane, 2 = pruned (plan.h)
    // Speculative extent (galario_b200.cu: run_call; the SPEC instantiation of the TMA kernel).  The transform of this
    // call was pruned to the extent the PREVIOUS call derived; this kernel verifies every point against it (ext_check,
    // viol), reduces max(u^2 + v^2) of ITS points as a by-product of the pass it makes over u and v anyway, and its
    // last CTA turns that into the extent for the next call (spec_out) and raises `redo` if a point lay outside: the
    // conditional second pass (fft.cuh / sample.cuh: redo_kernel, which leaves at once otherwise) then repeats
    // transform and sampling on spec_out, which covers every point by construction.
    unsigned long long* r2max;    // atomicMax of the bit pattern of u^2 + v^2 (SPEC only)
    int* spec_out;                // [3] not null: the last CTA writes the extent derived from r2max here and re-arms r2max
    unsigned int* redo;           // raised by the last CTA when viol != 0
    int* used_ext;                // [3] the extent the final result was computed with (gal_last_uv_extent)
};

// Which layout did the column pass write?  Same rule as fft.cuh: extent_is_whole_plane.
// Extents are produced on the device earlier in the same programmatic-launch chain (uv-extent kernel, the previous
// call's sampler): they are read only AFTER pdl_wait() and with L2-coherent loads (ld.global.cg), never through the
// non-coherent path, whose L1 line could predate the producer's store.
__device__ __forceinline__ bool extent_is_whole(const int* ext, int N) {
    return __ldcg(ext) >= N / 2 && __ldcg(ext + 1) <= 0 && __ldcg(ext + 2) >= N - 1;
}
// ... and which layout the column pass wrote (fft.cuh: layout_is_single, the same rule)
__device__ __forceinline__ bool layout_single(const int* ext, int N) {
#ifdef GAL_FORCE_PAIR
    return false;
#else
    return extent_is_whole(ext, N);
#endif
}

// Correctly rounded a / b from r = RN(1/b) (Markstein): q0 = RN(a r); rem = a - q0 b (exact in an
// FMA); q = RN(q0 + rem r).  Bit-identical to __ddiv_rn for the operand ranges met here (finite,
// normal, b without an all-ones significand — the host checks b and otherwise asks for a true
// division, EXACT).
template <bool EXACT>
__device__ __forceinline__ double div_by(double a, const IndexScalars& s) {
    if (EXACT) return s.du_exact_div ? __ddiv_rn(a, s.du) : __fma_rn(__fma_rn(-__dmul_rn(a, s.rdu), s.du, a), s.rdu, __dmul_rn(a, s.rdu));
    const double q0 = __dmul_rn(a, s.rdu);
    const double rem = __fma_rn(-q0, s.du, a);
    return __fma_rn(rem, s.rdu, q0);
}

// The listing's index arithmetic for one point (Eq. 11-12, 676-683), shared by the
// sampler and the uv-extent kernel so both take the same integer decisions.
struct PointIndex {
    double urot, vrot, uidx, vidx;
    bool uneg;
};
template <bool EXACT>
__device__ __forceinline__ PointIndex point_index(const IndexScalars& s, double u, double v) {
    PointIndex q;
    q.urot = __dsub_rn(__dmul_rn(u, s.cos_PA), __dmul_rn(v, s.sin_PA));
    q.vrot = __dadd_rn(__dmul_rn(u, s.sin_PA), __dmul_rn(v, s.cos_PA));
    q.uidx = div_by<EXACT>(fabs(q.urot), s);
    q.uneg = q.urot < 0.0;
    const double vq = div_by<EXACT>(q.vrot, s);
    // N/2 - v'/du where u' < 0 is N/2 + (-(v'/du)) bit for bit: flip the sign bit instead of selecting
    // (the comparison decides, not the sign bit of u': -0.0 takes the non-negative branch, reading A8)
    const double vs = __hiloint2double(__double2hiint(vq) ^ (q.uneg ? (int)0x80000000 : 0), __double2loint(vq));
    q.vidx = __dadd_rn(s.fH, vs);
    return q;
}
// the interpolation cell lies fully inside the stored half-plane grid
__device__ __forceinline__ bool cell_inside(const IndexScalars& s, const PointIndex& q) {
    return q.uidx <= s.fHm1 && q.vidx >= 0.0 && q.vidx < s.fN1;
}

// floor() and sincos() without the XU pipe.  On sm_100 the 64-bit conversions (FRND.F64, F2I.F64, I2F.F64)
// issue on the XU pipe at a small fraction of the FP64 rate; with two floors, two conversions and the
// range reduction of sincospi per point that pipe, not memory, bounded the sampler (ncu: XU 95 % busy).
// Both are therefore done with plain FP64 adds and integer bit moves.
//
// The constants of both routines live in constant memory so that each FP64 instruction reads its constant
// as a constant-bank operand; as literals they cost two uniform-register moves apiece, per point.
// [0..5] sine, [6..11] cosine kernel coefficients (fdlibm), then 1.5 * 2^52, pi / 2, 2^52.
static __constant__ double SINCOS_COEF[16] = {
    1.58969099521155010221e-10, -2.50507602534068634195e-08, 2.75573137070700676789e-06,
    -1.98412698298579493134e-04, 8.33333333332248946124e-03, -1.66666666666666324348e-01,
    -1.13596475577881948265e-11, 2.08757232129817482790e-09, -2.75573143513906633035e-07,
    2.48015872894767294178e-05, -1.38888888888741095749e-03, 4.16666666666666019037e-02,
    6755399441055744.0 /* 1.5 * 2^52: keeps negative k in range */, 1.57079632679489661923, 4503599627370496.0 /* 2^52 */, 0.0};

//
// floor of 0 <= x < 2^31 as a double (*fl) and as an int (return): x + 2^52 in round-down mode leaves floor(x) in
// the low mantissa bits.  fl is exactly floor(x), so the fractional weight x - fl is bit-identical to the
// listing's.  (Values outside that range give a meaningless result, never a trap: callers discard it.)
__device__ __forceinline__ int floor_small(double x, double* fl) {
    const double MAGIC = SINCOS_COEF[14];                // 2^52 (constant-bank operand)
    const double t = __dadd_rd(x, MAGIC);                // rounded towards -inf: exactly floor(x) + 2^52, no fix-up
    *fl = __dsub_rn(t, MAGIC);
    return __double2loint(t);
}

// sin and cos of 2 pi t for t in turns, |t| < 2^49.  k = rint(4 t) from the same mantissa trick (exact), the
// remainder r = 4 t - k in [-1/2, 1/2] is exact, a = r pi / 2 lies in [-pi/4, pi/4] where the classic
// minimax polynomials (fdlibm's kernel coefficients) are good to < 1 ulp; the quadrant k mod 4 then swaps and
// signs the pair.
// In _f32 (every array stored as float, tolerance 1e-4 of the peak) only the reduction stays in double — it
// is what keeps the phase of a 1e7-wavelength baseline exact — and the polynomials run in float.
__device__ __forceinline__ double quarter_reduce(double t, int* q) {
    const double* K = SINCOS_COEF;
    const double t4 = 4.0 * t;
    const double z = __dadd_rn(t4, K[12]);
    *q = __double2loint(z);
    return (t4 - (z - K[12])) * K[13];
}
__device__ __forceinline__ void sincos_quarter(double a, int q, double* sn, double* cs) {
    const double* K = SINCOS_COEF;
    const double a2 = a * a;
    double ps = K[0];
    ps = fma(ps, a2, K[1]);
    ps = fma(ps, a2, K[2]);
    ps = fma(ps, a2, K[3]);
    ps = fma(ps, a2, K[4]);
    ps = fma(ps, a2, K[5]);
    const double s = fma(a * a2, ps, a);
    double pc = K[6];
    pc = fma(pc, a2, K[7]);
    pc = fma(pc, a2, K[8]);
    pc = fma(pc, a2, K[9]);
    pc = fma(pc, a2, K[10]);
    pc = fma(pc, a2, K[11]);
    const double c = fma(a2 * a2, pc, fma(a2, -0.5, 1.0));
    const double ss = (q & 1) ? c : s, cc = (q & 1) ? s : c;
    *sn = (q & 2) ? -ss : ss;
    *cs = ((q + 1) & 2) ? -cc : cc;
}
__device__ __forceinline__ void sincos_quarter(float a, int q, float* sn, float* cs) {
    const float a2 = a * a;                       // single-precision kernels on [-pi/4, pi/4]: error < 1e-7
    float ps = 2.7557314297e-06f;
    ps = fmaf(ps, a2, -1.9841270114e-04f);
    ps = fmaf(ps, a2, 8.3333337680e-03f);
    ps = fmaf(ps, a2, -1.6666667163e-01f);
    const float s = fmaf(a * a2, ps, a);
    float pc = 2.4801587642e-05f;
    pc = fmaf(pc, a2, -1.3888889225e-03f);
    pc = fmaf(pc, a2, 4.1666667908e-02f);
    const float c = fmaf(a2 * a2, pc, fmaf(a2, -0.5f, 1.0f));
    const float ss = (q & 1) ? c : s, cc = (q & 1) ? s : c;
    *sn = (q & 2) ? -ss : ss;
    *cs = ((q + 1) & 2) ? -cc : cc;
}

// Node (kv mod N, ku mod N) of the spectrum extended to all integers by the periodicity and Hermitian symmetry
// of the DFT of a real image (reading A6): columns 0..N/2 are stored; column cu > N/2 is the conjugate of column
// N - cu at row -kv.  Used for the points whose cell leaves the half-plane grid; 32-bit index arithmetic.
template <typename T, bool PAIR>
__device__ __forceinline__ cx<T> node_wrapped(const NodePair<T>* __restrict__ spec, int N, int cu, int kvm) {
    const int H = N >> 1, m = N - 1;
    auto at = [&](int e) -> cx<T> {
        return PAIR ? __ldg(&spec[e].a) : __ldg(reinterpret_cast<const cx<T>*>(spec) + e);
    };
    if (cu <= H) return at(cu * N + ((kvm + H) & m));
    cx<T> g = at((N - cu) * N + (((N - kvm) + H) & m));
    g.y = -g.y;
    return g;
}

// Bilinear interpolation of the extended spectrum at (uidx, vidx) anywhere in the plane: the listing's
// interpolation on wrapped nodes.  Out of line: one call per out-of-grid point keeps the hot
// loop of the sampler free of this code.
template <typename T, bool PAIR>
__device__ __noinline__ cx<double> wrapped_cell(const NodePair<T>* __restrict__ spec, int N, double uidx, double vidx) {
    const double fx = floor(uidx), fy = floor(vidx);
    const long long ix = (long long)fx, iy = (long long)fy;
    const int m = N - 1, H = N >> 1;                        // N is a power of two: & m is the floor-mod
    const int c0 = (int)(ix & m), c1 = (int)((ix + 1) & m);
    const int kv0 = (int)((iy - H) & m), kv1 = (int)((iy + 1 - H) & m);
    const cx<T> g00 = node_wrapped<T, PAIR>(spec, N, c0, kv0), g01 = node_wrapped<T, PAIR>(spec, N, c1, kv0);
    const cx<T> g10 = node_wrapped<T, PAIR>(spec, N, c0, kv1), g11 = node_wrapped<T, PAIR>(spec, N, c1, kv1);
    const double txr = __dsub_rn(uidx, fx), tyr = __dsub_rn(vidx, fy);
    const double ax = 1.0 - txr, ay = 1.0 - tyr;
    cx<double> r;
    r.x = ay * (ax * (double)g00.x + txr * (double)g01.x) + tyr * (ax * (double)g10.x + txr * (double)g11.x);
    r.y = ay * (ax * (double)g00.y + txr * (double)g01.y) + tyr * (ax * (double)g10.y + txr * (double)g11.y);
    return r;
}

// ------------------------------------------------------------------------------------------
// uv extent: which part of the half plane can the point set reach?
// ext[0] = largest column ku any interpolation cell touches, ext[1] / ext[2] = smallest / largest
// shifted row kvs; a point whose cell leaves the grid (reading A6: the wrap can reach anything)
// sets the full extent.  Integer max/min only, so the result does not depend on the order.
// The FFT passes skip what lies outside (fft.cuh), which changes no result.
// Pure streaming (16 B per point): EU points per thread are requested before any arithmetic.
// ------------------------------------------------------------------------------------------
struct ExtentParams {
    int N;
    long long total;       // C * M
    IndexScalars ix;
    int* ext;              // [3], initialised by the host to the cell of the sampler's dead slots
};

// Every step of the index arithmetic after the rotation is monotone in its argument (a correctly rounded
// division by du > 0, a rounded addition to N/2, floor), so the extremes of the indices are the indices of
// the extremes: the loop only tracks max |u'| and min / max of the signed v term (v' where u' >= 0, -v'
// where u' < 0 — the listing's N/2 - v'/du equals N/2 + (-v')/du bit for bit) and the divisions, the floor and
// the inside-the-grid test are applied once per warp to those three numbers.
template <typename T>
__global__ void __launch_bounds__(256, 4) uv_extent_kernel(const ExtentParams p, const T* __restrict__ u,
                                                           const T* __restrict__ v) {
    // Persistent grid (a whole number of CTAs per SM), EU points per thread and trip; the loads of the next
    // trip are issued before the arithmetic of this one (register double buffer).
    constexpr int EU = 4;
    const int N = p.N, H = N >> 1;
    double umax = 0.0, smin = 0.0, smax = 0.0;               // (0, 0): the dead-slot cell, always in the extent
    pdl_wait();
    const long long stride = (long long)gridDim.x * blockDim.x * EU;
    long long k0 = (long long)blockIdx.x * blockDim.x * EU + threadIdx.x;
    double nu[EU], nv[EU];
    auto fetch = [&](long long kk) {
#pragma unroll
        for (int j = 0; j < EU; ++j) {
            const long long k = kk + j * 256;
            const bool ok = k < p.total;
            nu[j] = ok ? (double)__ldcs(u + k) : 0.0;
            nv[j] = ok ? (double)__ldcs(v + k) : 0.0;
        }
    };
    fetch(k0);
    for (; k0 < p.total; k0 += stride) {
        double pu[EU], pv[EU];
#pragma unroll
        for (int j = 0; j < EU; ++j) { pu[j] = nu[j]; pv[j] = nv[j]; }
        fetch(k0 + stride);
#pragma unroll
        for (int j = 0; j < EU; ++j) {
            const double urot = __dsub_rn(__dmul_rn(pu[j], p.ix.cos_PA), __dmul_rn(pv[j], p.ix.sin_PA));
            const double vrot = __dadd_rn(__dmul_rn(pu[j], p.ix.sin_PA), __dmul_rn(pv[j], p.ix.cos_PA));
            const double sv = urot < 0.0 ? -vrot : vrot;
            umax = fmax(umax, fabs(urot));
            smin = fmin(smin, sv);
            smax = fmax(smax, sv);
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        umax = fmax(umax, __shfl_xor_sync(0xffffffffu, umax, o));
        smin = fmin(smin, __shfl_xor_sync(0xffffffffu, smin, o));
        smax = fmax(smax, __shfl_xor_sync(0xffffffffu, smax, o));
    }
    // one set of atomics per CTA: same-address atomics serialise in L2 and would otherwise be the kernel's tail
    __shared__ double red[3][8];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    if (lane == 0) { red[0][wid] = umax; red[1][wid] = smin; red[2][wid] = smax; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int i = 1; i < 8; ++i) {
            umax = fmax(umax, red[0][i]); smin = fmin(smin, red[1][i]); smax = fmax(smax, red[2][i]);
        }
        PointIndex lo, hi;                                    // the two extreme cells of this CTA's points
        lo.uidx = hi.uidx = div_by<false>(umax, p.ix);
        lo.vidx = __dadd_rn(p.ix.fH, div_by<false>(smin, p.ix));
        hi.vidx = __dadd_rn(p.ix.fH, div_by<false>(smax, p.ix));
        int cmax = H, rmin = 0, rmax = N - 1;                 // a cell leaves the grid: everything (reading A6)
        if (cell_inside(p.ix, lo) && cell_inside(p.ix, hi)) {
            cmax = (int)floor(hi.uidx) + 1;
            rmin = (int)floor(lo.vidx);
            rmax = (int)floor(hi.vidx) + 1;
        }
        atomicMax(p.ext + 0, cmax);
        atomicMin(p.ext + 1, rmin);
        atomicMax(p.ext + 2, rmax);
    }
}

// Points per thread and tile (U), stages of the shared-memory ring, resident CTAs per SM the register
// budget is set for.
#ifndef GAL_SAMPLE_U32
#define GAL_SAMPLE_U32 2             // points per thread and tile in fp32
#endif
#ifndef GAL_SAMPLE_U
#define GAL_SAMPLE_U 2
#endif
#ifndef GAL_SAMPLE_STAGES
#define GAL_SAMPLE_STAGES 3
#endif
#ifndef GAL_SAMPLE_MINB
#define GAL_SAMPLE_MINB 2
#endif
#ifndef GAL_SAMPLE_NT
#define GAL_SAMPLE_NT 256            // consumer threads per CTA
#endif

// The unit of work is a tile of 256*U consecutive points; CTA b takes tiles b, b + gridDim.x, ...; thread t
// of the 256 consumer threads takes points t, t + 256, ... of the tile.
template <typename T, bool DO_CHI2> struct SampleGeom {
    static constexpr int U = sizeof(T) == 4 ? GAL_SAMPLE_U32 : GAL_SAMPLE_U;
    static constexpr int NT = GAL_SAMPLE_NT, NW = NT / 32;         // consumer threads / warps
    static constexpr int NT_TMA = NT + 32;                          // + one producer warp (TMA kernel)
    static constexpr int TILE = NT * U;
    static constexpr int NARR = DO_CHI2 ? 5 : 2;
    static constexpr int S = GAL_SAMPLE_STAGES;
    static constexpr uint32_t ARR_BYTES = TILE * sizeof(T);         // multiple of 16
    static constexpr uint32_t STAGE_BYTES = NARR * ARR_BYTES;
    static constexpr size_t SMEM = (size_t)S * STAGE_BYTES + 16 * S;
};

// One column-pair entry through the read-only path: a single 256-bit load in fp64 (sm_100), 128-bit in fp32.
__device__ __forceinline__ NodePair<double> load_pair(const NodePair<double>* p) {
    NodePair<double> e;
    asm("ld.global.nc.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(e.a.x), "=d"(e.a.y), "=d"(e.b.x), "=d"(e.b.y) : "l"(p));
    return e;
}
__device__ __forceinline__ NodePair<float> load_pair(const NodePair<float>* p) {
    const float4 q = __ldg(reinterpret_cast<const float4*>(p));
    NodePair<float> e;
    e.a.x = q.x; e.a.y = q.y; e.b.x = q.z; e.b.y = q.w;
    return e;
}

// What every variant of the kernel needs per CTA.
template <typename T> struct SampleCtx {
    const NodePair<T>* spec;   // this channel's spectrum
    int N;
    int odd;               // lane parity
    double acc;            // chi2 partial of this thread
    unsigned int oob;      // points of this thread beyond the half-plane grid
    unsigned int viol;     // points of this thread outside the extent of the bound uv set
    int ck_kumax, ck_rmin, ck_rmax;   // that extent ({N, 0, N}: nothing to check)
    double r2;             // largest u^2 + v^2 of this thread's points (SPEC)
};

// Everything after the interpolation of one point: sign for u' < 0, phase, store / chi2 term.
template <typename T, bool WRITE_VIS, bool DO_CHI2>
__device__ __forceinline__ void point_tail(const SampleParams<T>& p, SampleCtx<T>& cx_, T ReInt, T ImInt, bool uneg, double turns,
                                           long long k, long long M, int c, T re_obs, T im_obs, T w) {
    using R = T;
    if (uneg) ImInt = -ImInt;
    R vr = ReInt, vi = ImInt;
    if (p.has_phase) {
        int qd;
        const double a = quarter_reduce(turns, &qd);
        R sn, co;
        sincos_quarter((R)a, qd, &sn, &co);
        vr = ReInt * co - ImInt * sn;
        vi = ReInt * sn + ImInt * co;
    }
    if (p.amp != 1.0) { vr *= (R)p.amp; vi *= (R)p.amp; }
    if (WRITE_VIS) {
        if (k < M) {
            cx<T>* dst = reinterpret_cast<cx<T>*>(p.vis) + c * M + k;
            if (p.accumulate) { const cx<T> old = *dst; vr += old.x; vi += old.y; }
            __stcs(dst, mk<T>(vr, vi));
        }
    }
    if (DO_CHI2) {                                          // PAPER.md:718 (Eq. 10); w = 0 for dead slots
        const R dr = vr - re_obs;
        const R di = vi - im_obs;
        cx_.acc += (double)(fma(dr, dr, di * di) * w);
    }
}

// U points of one thread: rotate, index, gather, interpolate, phase, chi2 / store.
//   ld(a, j): value a (0 = u, 1 = v, 2 = re_obs, 3 = im_obs, 4 = w) of this thread's j-th point;
//             points past the end read as u = v = 0 with weight 0 (cell (0, N/2), always inside).
//   kpt(j):   global index of that point (only used to store the visibility).
//
// Gather by lane pairs.  The four nodes of a cell are two adjacent column-pair entries, (ku, kvs) and
// (ku, kvs+1): 64 contiguous bytes in fp64.  What bounds the gather is the L2 -> SM path (about 43 bytes
// per clock and SM, measured) and the L1's one line per clock, so the access is shaped to move the fewest
// sectors and lines: lanes 2i and 2i+1 fetch each other's cells together — in each of the two load
// instructions the even lane reads entry kvs and the odd lane entry kvs+1 of the SAME cell with one
// 256-bit load (two sectors, 1.25 lines per cell; measured 45 clk per 32 points against 72 for the
// single-copy layout and 126 for one 16-byte load per node and lane).  Each lane then interpolates its row
// along u for both cells, one shuffle hands the row the partner needs across, and the owner finishes its
// own point.
template <typename T, bool WRITE_VIS, bool DO_CHI2, bool EXACT, int U, bool PAIR, bool SPEC = false, typename LD, typename KP>
__device__ __forceinline__ void sample_points(const SampleParams<T>& p, SampleCtx<T>& cx_, LD ld, KP kpt, long long M,
                                              int c) {
    const int N = cx_.N, odd = cx_.odd;
    const NodePair<T>* __restrict__ spec = cx_.spec;
    using R = T;                            // type of the value arithmetic (interpolation, phase product, chi2 terms)
    R tx[U], ty[U], tx_partner[U];
    double turns[U];
    bool uneg[U], inside[U];
    cx<T> ga0[U], ga1[U], gb0[U], gb1[U];   // even lane's cell (a) / odd lane's cell (b); column ku+0 / ku+1
#pragma unroll
    for (int j = 0; j < U; ++j) {
        const PointIndex q = point_index<EXACT>(p.ix, (double)ld(0, j), (double)ld(1, j));
        if (SPEC) cx_.r2 = fmax(cx_.r2, fma(q.urot, q.urot, q.vrot * q.vrot));               // = u^2 + v^2 up to rounding (margin in the verdict)
        // bilinear interpolation
        inside[j] = cell_inside(p.ix, q);
        uneg[j] = q.uneg;
        double fx0, fy0;
        const int ix0 = floor_small(q.uidx, &fx0), iy0 = floor_small(q.vidx, &fy0);      // (meaningless outside the grid)
        tx[j] = (R)__dsub_rn(q.uidx, fx0);               // (outside the grid the rare path below redoes this)
        ty[j] = (R)__dsub_rn(q.vidx, fy0);
        // theta / 2 pi in turns (exact range reduction in quarter_reduce)
        turns[j] = fma(q.urot, p.dRA_turns, q.vrot * p.dDec_turns);
        const int off = inside[j] ? ix0 * N + iy0 : 0;   // outside the grid: any valid entry (the rare path below redoes the point)
        if (ix0 + 1 > cx_.ck_kumax || iy0 < cx_.ck_rmin || iy0 + 1 > cx_.ck_rmax || (!inside[j] && cx_.ck_kumax < N)) ++cx_.viol;
        const int off_partner = __shfl_xor_sync(0xffffffffu, off, 1);
        const int ia = (odd ? off_partner : off) + odd, ib = (odd ? off : off_partner) + odd;
        if (PAIR) {
            const NodePair<T> ea = load_pair(spec + ia);
            const NodePair<T> eb = load_pair(spec + ib);
            ga0[j] = ea.a; ga1[j] = ea.b;
            gb0[j] = eb.a; gb1[j] = eb.b;
        } else {                    // single-copy layout: the same four values from columns ku and ku + 1
            const cx<T>* __restrict__ sg = reinterpret_cast<const cx<T>*>(spec);
            ga0[j] = __ldg(sg + ia); ga1[j] = __ldg(sg + ia + N);
            gb0[j] = __ldg(sg + ib); gb1[j] = __ldg(sg + ib + N);
        }
        tx_partner[j] = __shfl_xor_sync(0xffffffffu, tx[j], 1);     // in flight with the gather
    }
#pragma unroll
    for (int j = 0; j < U; ++j) {
        const R txa = odd ? tx_partner[j] : tx[j], txb = odd ? tx[j] : tx_partner[j];
        // this lane's row (kvs + odd) of both cells, interpolated along u: g0 + t (g1 - g0)
        const R ra_re = fma(txa, ga1[j].x - ga0[j].x, ga0[j].x);
        const R ra_im = fma(txa, ga1[j].y - ga0[j].y, ga0[j].y);
        const R rb_re = fma(txb, gb1[j].x - gb0[j].x, gb0[j].x);
        const R rb_im = fma(txb, gb1[j].y - gb0[j].y, gb0[j].y);
        // the even lane keeps row kvs of cell a and needs row kvs+1 of it; the odd lane keeps row kvs+1 of
        // cell b and needs row kvs: mine + w (other - mine), w = ty (even) or 1 - ty (odd)
        const R o_re = __shfl_xor_sync(0xffffffffu, odd ? ra_re : rb_re, 1);
        const R o_im = __shfl_xor_sync(0xffffffffu, odd ? ra_im : rb_im, 1);
        const R m_re = odd ? rb_re : ra_re, m_im = odd ? rb_im : ra_im;
        const R wy = odd ? (R)1 - ty[j] : ty[j];
        R ReInt = fma(wy, o_re - m_re, m_re);
        R ImInt = fma(wy, o_im - m_im, m_im);
        if (!inside[j]) {           // rare: the cell leaves the half-plane grid (reading A6); dead slots never get here
            const PointIndex q = point_index<EXACT>(p.ix, (double)ld(0, j), (double)ld(1, j));
            if (q.uidx > p.ix.fH || q.vidx < 0.0 || q.vidx > p.ix.fN1) ++cx_.oob;
            const cx<double> g = wrapped_cell<T, PAIR>(spec, N, q.uidx, q.vidx);
            ReInt = (R)g.x;
            ImInt = (R)g.y;
        }
        point_tail<T, WRITE_VIS, DO_CHI2>(p, cx_, ReInt, ImInt, uneg[j], turns[j], kpt(j), M, c, ld(2, j), ld(3, j), ld(4, j));
    }
}

// The same U points with every thread gathering its OWN cell (two entries of the pair layout / four values of the
// single-copy layout), no lane pairing: fewer instructions (no shuffles, no selects) but one L1 line per lane and
// load instead of one per lane pair.  Taken for a bound observation set (gal_plan_bind_obs), whose uv-sorted
// order makes the lanes of a warp share their lines; in time-major order it loses to the lane-pair gather.
template <typename T, bool WRITE_VIS, bool DO_CHI2, bool EXACT, int U, bool PAIR, typename LD, typename KP>
__device__ __forceinline__ void sample_points_direct(const SampleParams<T>& p, SampleCtx<T>& cx_, LD ld, KP kpt, long long M,
                                                     int c) {
    const int N = cx_.N;
    const NodePair<T>* __restrict__ spec = cx_.spec;
    using R = T;
    R tx[U], ty[U];
    double turns[U];
    bool uneg[U], inside[U];
    cx<T> g00[U], g01[U], g10[U], g11[U];                   // g[row kvs + 0/1][column ku + 0/1]
#pragma unroll
    for (int j = 0; j < U; ++j) {
        const PointIndex q = point_index<EXACT>(p.ix, (double)ld(0, j), (double)ld(1, j));
        inside[j] = cell_inside(p.ix, q);
        uneg[j] = q.uneg;
        double fx0, fy0;
        const int ix0 = floor_small(q.uidx, &fx0), iy0 = floor_small(q.vidx, &fy0);      // (meaningless outside the grid)
        tx[j] = (R)__dsub_rn(q.uidx, fx0);
        ty[j] = (R)__dsub_rn(q.vidx, fy0);
        turns[j] = fma(q.urot, p.dRA_turns, q.vrot * p.dDec_turns);
        const int off = inside[j] ? ix0 * N + iy0 : 0;
        if (ix0 + 1 > cx_.ck_kumax || iy0 < cx_.ck_rmin || iy0 + 1 > cx_.ck_rmax || (!inside[j] && cx_.ck_kumax < N)) ++cx_.viol;
        if (PAIR) {
            const NodePair<T> e0 = load_pair(spec + off), e1 = load_pair(spec + off + 1);
            g00[j] = e0.a; g01[j] = e0.b; g10[j] = e1.a; g11[j] = e1.b;
        } else {
            const cx<T>* __restrict__ sg = reinterpret_cast<const cx<T>*>(spec);
            g00[j] = __ldg(sg + off); g10[j] = __ldg(sg + off + 1);
            g01[j] = __ldg(sg + off + N); g11[j] = __ldg(sg + off + N + 1);
        }
    }
#pragma unroll
    for (int j = 0; j < U; ++j) {
        // along u in both rows, then along v
        const R r0_re = fma(tx[j], g01[j].x - g00[j].x, g00[j].x), r0_im = fma(tx[j], g01[j].y - g00[j].y, g00[j].y);
        const R r1_re = fma(tx[j], g11[j].x - g10[j].x, g10[j].x), r1_im = fma(tx[j], g11[j].y - g10[j].y, g10[j].y);
        R ReInt = fma(ty[j], r1_re - r0_re, r0_re);
        R ImInt = fma(ty[j], r1_im - r0_im, r0_im);
        if (!inside[j]) {           // rare: the cell leaves the half-plane grid (reading A6)
            const PointIndex q = point_index<EXACT>(p.ix, (double)ld(0, j), (double)ld(1, j));
            if (q.uidx > p.ix.fH || q.vidx < 0.0 || q.vidx > p.ix.fN1) ++cx_.oob;
            const cx<double> g = wrapped_cell<T, PAIR>(spec, N, q.uidx, q.vidx);
            ReInt = (R)g.x;
            ImInt = (R)g.y;
        }
        point_tail<T, WRITE_VIS, DO_CHI2>(p, cx_, ReInt, ImInt, uneg[j], turns[j], kpt(j), M, c, ld(2, j), ld(3, j), ld(4, j));
    }
}

// Deterministic reduction: warp shuffle -> block -> per-block partial -> last block (ticket), fixed order,
// no floating-point atomics.  Also adds this CTA's out-of-grid count.
template <typename T, bool DO_CHI2>
__device__ __forceinline__ void sample_finish(const SampleParams<T>& p, int c, double acc, unsigned int oob,
                                              unsigned int viol, double r2 = 0.0) {
    if (p.ext_check) {                                       // a bound uv set or a speculative extent is being verified
        viol = __reduce_add_sync(0xffffffffu, viol);
        if ((threadIdx.x & 31) == 0 && viol) {
            atomicAdd(p.viol, (unsigned long long)viol);
            if (p.viol_flag) *(volatile unsigned int*)p.viol_flag = 1u;
        }
    }
    if (p.spec_out) {                                        // bit patterns of non-negative doubles order like integers
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) r2 = fmax(r2, __shfl_xor_sync(0xffffffffu, r2, o));
        if ((threadIdx.x & 31) == 0) atomicMax(p.r2max, (unsigned long long)__double_as_longlong(r2));
    }
    __shared__ double wsum[32];
    __shared__ unsigned int woob[32];
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
        if (p.spec_out) __threadfence();                        // this CTA's atomics before its ticket
        // the last CTA of the launch re-arms the state of the next call: counter 0, extent = the dead-slot cell
        if (atomicAdd(p.done, 1u) == gridDim.x * gridDim.y - 1) {
            if (p.spec_out) {                                   // speculative extent: by-product and verdict (SampleParams)
                __threadfence();
                const unsigned long long bits = atomicExch(p.r2max, 0ull);          // read and re-arm
                const double imax = sqrt(__longlong_as_double((long long)bits)) * (1.0 + 1e-12) / p.ix.du;
                const int H = p.N / 2;
                int e0 = H, e1 = 0, e2 = p.N - 1;               // as extent_from_radius_kernel: two cells of margin
                if (imax + 3.0 < (double)(H - 1)) {
                    const int k = (int)imax + 2;
                    e0 = k + 1; e1 = H - k - 1; e2 = H + k + 1;
                }
                p.spec_out[0] = e0; p.spec_out[1] = e1; p.spec_out[2] = e2;
                // (a whole-plane extent covers every point, wrapped ones too: it cannot fail)
                const bool failed = p.ext_check && !extent_is_whole(p.ext_check, p.N) && atomicAdd(p.viol, 0ull) != 0ull;
                if (failed) { *p.redo = 1u; atomicExch(p.oob, 0ull); }              // the second pass counts again
                p.used_ext[0] = failed ? e0 : __ldcg(p.ext);
                p.used_ext[1] = failed ? e1 : __ldcg(p.ext + 1);
                p.used_ext[2] = failed ? e2 : __ldcg(p.ext + 2);
            }
            if (p.rearm) {
                int* nx = reinterpret_cast<int*>(p.next_state);
                nx[0] = 0; nx[1] = 0;
                nx[2] = 1; nx[3] = p.N / 2; nx[4] = p.N / 2 + 1;
                nx[5] = 0;                                      // its own done ticket
                nx[6] = 0; nx[7] = 0;                           // and its extent-violation counter
            }
            *p.done = 0;
            if (p.ext_hint && p.ext) *(volatile unsigned int*)p.ext_hint = extent_is_whole(p.ext, p.N) ? 1u : 2u;
        }
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

// One tile by plain (guarded) loads straight from global memory.
template <typename T, bool WRITE_VIS, bool DO_CHI2, bool EXACT, bool PAIR, bool SPEC = false>
__device__ __forceinline__ void sample_tile_plain(const SampleParams<T>& p, SampleCtx<T>& cx_, long long tile, long long M,
                                                  int c) {
    constexpr int U = SampleGeom<T, DO_CHI2>::U, TILE = SampleGeom<T, DO_CHI2>::TILE;
    const long long k0 = tile * TILE + threadIdx.x;
    const T* __restrict__ g0 = p.u + c * M;
    const T* __restrict__ g1 = p.v + c * M;
    const T* __restrict__ g2 = DO_CHI2 ? p.re_obs + c * M : nullptr;
    const T* __restrict__ g3 = DO_CHI2 ? p.im_obs + c * M : nullptr;
    const T* __restrict__ g4 = DO_CHI2 ? p.w + c * M : nullptr;
    auto ld = [&](int a, int j) -> T {
        const long long k = k0 + j * GAL_SAMPLE_NT;
        if (k >= M) return (T)0;
        const T* g = a == 0 ? g0 : a == 1 ? g1 : a == 2 ? g2 : a == 3 ? g3 : g4;
        return __ldcs(g + k);
    };
    auto kpt = [&](int j) -> long long { return k0 + j * GAL_SAMPLE_NT; };
    sample_points<T, WRITE_VIS, DO_CHI2, EXACT, U, PAIR, SPEC>(p, cx_, ld, kpt, M, c);
}

template <typename T>
__device__ __forceinline__ SampleCtx<T> sample_ctx(const SampleParams<T>& p, int c) {
    SampleCtx<T> cx_;
    cx_.N = p.N;
    // channel c of the batch: [N/2+1][N] entries, column pairs or (whole-plane extent) single values
    const long long plane = p.shared_spec ? 0ll : (long long)c * (p.N / 2 + 1) * p.N;
    cx_.spec = layout_single(p.ext, p.N) ? reinterpret_cast<const NodePair<T>*>(reinterpret_cast<const cx<T>*>(p.spec) + plane)
                                           : p.spec + plane;
    cx_.odd = threadIdx.x & 1;
    cx_.acc = 0.0;
    cx_.oob = 0;
    cx_.viol = 0;
    cx_.r2 = 0.0;
    cx_.ck_kumax = p.N; cx_.ck_rmin = 0; cx_.ck_rmax = p.N;
    if (p.ext_check) { cx_.ck_kumax = __ldcg(p.ext_check); cx_.ck_rmin = __ldcg(p.ext_check + 1); cx_.ck_rmax = __ldcg(p.ext_check + 2); }
    return cx_;
}

// General kernel (256 threads): any alignment, any du (takes the true division when the shortcut is not valid).
template <typename T, bool WRITE_VIS, bool DO_CHI2>
__global__ void __launch_bounds__(GAL_SAMPLE_NT, GAL_SAMPLE_MINB) sample_kernel_plain(const SampleParams<T> p) {
    using G = SampleGeom<T, DO_CHI2>;
    const int c = blockIdx.y;
    const long long M = p.M;
    pdl_wait();
    SampleCtx<T> cx_ = sample_ctx(p, c);                     // (reads the extent: after the wait)
    const long long ntiles = (M + G::TILE - 1) / G::TILE;
    if (layout_single(p.ext, p.N)) {
        for (long long tile = blockIdx.x; tile < ntiles; tile += gridDim.x)
            sample_tile_plain<T, WRITE_VIS, DO_CHI2, true, false>(p, cx_, tile, M, c);
    } else {
        for (long long tile = blockIdx.x; tile < ntiles; tile += gridDim.x)
            sample_tile_plain<T, WRITE_VIS, DO_CHI2, true, true>(p, cx_, tile, M, c);
    }
    sample_finish<T, DO_CHI2>(p, c, cx_.acc, cx_.oob, cx_.viol);
}

// Fast kernel (256 consumer threads + one producer warp): every per-point array 16-byte aligned in every
// channel, du fit for the division shortcut.  Warp specialisation: lane 0 of the ninth warp is the TMA
// producer — it waits for a stage to be released (`empty` mbarrier, one arrival per consumer warp), arms the
// `full` mbarrier with the byte count and issues the bulk copies of the next tile; the consumer warps wait on
// `full`, work, and release the stage.  No block-wide barrier in the loop: a consumer warp only ever waits
// for data, the producer runs up to S tiles ahead.  The ragged last tile (if any) is read with plain loads
// by the CTA whose turn it would have been.
template <typename T, bool WRITE_VIS, bool DO_CHI2, bool SPEC = false>
__global__ void __launch_bounds__(SampleGeom<T, DO_CHI2>::NT_TMA, GAL_SAMPLE_MINB) sample_kernel_tma(const SampleParams<T> p) {
    using G = SampleGeom<T, DO_CHI2>;
    constexpr int U = G::U, TILE = G::TILE, S = G::S;
    extern __shared__ __align__(128) unsigned char sample_smem[];
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int c = blockIdx.y;
    const long long M = p.M;
    const int nfull = (int)(M / TILE);
    const uint32_t stage0 = smem_u32(sample_smem);
    const uint32_t full0 = stage0 + S * G::STAGE_BYTES, empty0 = full0 + 8 * S;
    if (tid == 0) {
        for (int s = 0; s < S; ++s) { mbar_init(full0 + 8 * s, 1); mbar_init(empty0 + 8 * s, G::NW); }
        mbar_fence_init();
    }
    pdl_wait();
    __syncthreads();
    SampleCtx<T> cx_ = sample_ctx(p, c);                     // (reads the extent: after the wait)

    if (wid == G::NW) {
        if (lane == 0) {                                     // ---- producer ----
            const uint64_t pol = l2_policy_evict_first();
            uint32_t stage = 0, parity = 1;                  // a fresh mbarrier lets a wait on parity 1 through
            for (int tile = blockIdx.x; tile < nfull; tile += gridDim.x) {
                mbar_wait_relaxed(empty0 + 8 * stage, parity);
                const uint32_t mb = full0 + 8 * stage, dst = stage0 + stage * G::STAGE_BYTES;
                const long long k = (long long)tile * TILE + c * M;
                mbar_expect_tx(mb, G::STAGE_BYTES);
                tma_load_1d(dst, p.u + k, G::ARR_BYTES, mb, pol);
                tma_load_1d(dst + G::ARR_BYTES, p.v + k, G::ARR_BYTES, mb, pol);
                if (DO_CHI2) {
                    tma_load_1d(dst + 2 * G::ARR_BYTES, p.re_obs + k, G::ARR_BYTES, mb, pol);
                    tma_load_1d(dst + 3 * G::ARR_BYTES, p.im_obs + k, G::ARR_BYTES, mb, pol);
                    tma_load_1d(dst + 4 * G::ARR_BYTES, p.w + k, G::ARR_BYTES, mb, pol);
                }
                if (++stage == S) { stage = 0; parity ^= 1u; }
            }
        }
    } else {                                                 // ---- consumers ----
        auto consume = [&](auto pair_tag, auto direct_tag) { // the loop, once per spectrum layout and gather scheme
            constexpr bool PAIR = decltype(pair_tag)::value;
            constexpr bool DIRECT = decltype(direct_tag)::value;
            uint32_t stage = 0, parity = 0;
            int tile = blockIdx.x;
            for (; tile < nfull; tile += gridDim.x) {
                mbar_wait(full0 + 8 * stage, parity);
                const T* st = reinterpret_cast<const T*>(sample_smem + stage * G::STAGE_BYTES) + tid;
                auto ld = [&](int a, int j) -> T { return st[a * TILE + j * GAL_SAMPLE_NT]; };
                auto kpt = [&](int j) -> long long { return (long long)tile * TILE + j * GAL_SAMPLE_NT + tid; };
                if (DIRECT) sample_points_direct<T, WRITE_VIS, DO_CHI2, false, U, PAIR>(p, cx_, ld, kpt, M, c);
                else sample_points<T, WRITE_VIS, DO_CHI2, false, U, PAIR, SPEC>(p, cx_, ld, kpt, M, c);
                __syncwarp();                                // every lane has read its last value of this stage
                if (lane == 0) mbar_arrive(empty0 + 8 * stage);
                if (++stage == S) { stage = 0; parity ^= 1u; }
            }
            if (tile == nfull && (long long)nfull * TILE < M)    // the ragged last tile falls to this CTA
                sample_tile_plain<T, WRITE_VIS, DO_CHI2, false, PAIR, SPEC>(p, cx_, nfull, M, c);
        };
        const bool whole = layout_single(p.ext, p.N);
        if (!SPEC && DO_CHI2 && p.direct) {                  // (a bound observation set is a chi2 matter)
            if (whole) consume(std::false_type{}, std::true_type{}); else consume(std::true_type{}, std::true_type{});
        } else {
            if (whole) consume(std::false_type{}, std::false_type{}); else consume(std::true_type{}, std::false_type{});
        }
    }
    sample_finish<T, DO_CHI2>(p, c, cx_.acc, cx_.oob, cx_.viol, cx_.r2);
}

// ------------------------------------------------------------------------------------------
// Multi-source composition in ONE launch ("summing up the visibilities of each single source ...
// applying a different complex phase"): V(u, v) = sum_s amp_s V_s(u, v; PA_s, dRA_s, dDec_s)
// of ONE model spectrum.  The per-point arrays are read once, the S placements are looped inside the per-point
// routine (each one re-rotates the point and gathers its own cell), the sum is compared with the observations
// in the same kernel: no read-modify-write of vis, no scratch buffer, no second kernel.  One thread per point,
// plain loads (any alignment); the placements travel in the kernel parameter block.
// ------------------------------------------------------------------------------------------
template <typename T, bool PAIR>
__device__ __forceinline__ void multi_point(const SampleParams<T>& p, const PlacementSet& ps, const NodePair<T>* __restrict__ spec,
                                            double u, double v, double& vr, double& vi, unsigned int& oob,
                                            int ck_kumax, int ck_rmin, int ck_rmax, unsigned int& viol) {
    const int N = p.N;
    for (int s = 0; s < ps.S; ++s) {
        const Placement& pl = ps.pl[s];
        IndexScalars ix = p.ix;
        ix.cos_PA = pl.cos_PA; ix.sin_PA = pl.sin_PA;
        const PointIndex q = point_index<true>(ix, u, v);
        double re, im;
        if (cell_inside(ix, q)) {
            double fx0, fy0;
            const int ix0 = floor_small(q.uidx, &fx0), iy0 = floor_small(q.vidx, &fy0);
            const double tx = __dsub_rn(q.uidx, fx0), ty = __dsub_rn(q.vidx, fy0);
            const int off = ix0 * N + iy0;
            if (ix0 + 1 > ck_kumax || iy0 < ck_rmin || iy0 + 1 > ck_rmax) ++viol;   // outside the extent the transform was pruned to
            cx<T> g00, g01, g10, g11;                                         // g[row][column]
            if (PAIR) {
                const NodePair<T> e0 = load_pair(spec + off), e1 = load_pair(spec + off + 1);
                g00 = e0.a; g01 = e0.b; g10 = e1.a; g11 = e1.b;
            } else {
                const cx<T>* __restrict__ sg = reinterpret_cast<const cx<T>*>(spec);
                g00 = __ldg(sg + off); g10 = __ldg(sg + off + 1); g01 = __ldg(sg + off + N); g11 = __ldg(sg + off + N + 1);
            }
            const double r0r = fma(tx, (double)g01.x - (double)g00.x, (double)g00.x), r0i = fma(tx, (double)g01.y - (double)g00.y, (double)g00.y);
            const double r1r = fma(tx, (double)g11.x - (double)g10.x, (double)g10.x), r1i = fma(tx, (double)g11.y - (double)g10.y, (double)g10.y);
            re = fma(ty, r1r - r0r, r0r);
            im = fma(ty, r1i - r0i, r0i);
        } else {                                                              // reading A6
            if (q.uidx > ix.fH || q.vidx < 0.0 || q.vidx > ix.fN1) ++oob;
            if (ck_kumax < N) ++viol;                                         // (a wrapped cell needs the whole plane)
            const cx<double> g = wrapped_cell<T, PAIR>(spec, N, q.uidx, q.vidx);
            re = g.x; im = g.y;
        }
        if (q.uneg) im = -im;
        if (pl.has_phase) {
            int qd;
            const double a = quarter_reduce(fma(q.urot, pl.dRA_turns, q.vrot * pl.dDec_turns), &qd);
            double sn, co;
            sincos_quarter(a, qd, &sn, &co);
            const double t = re * co - im * sn;
            im = re * sn + im * co;
            re = t;
        }
        vr = fma(pl.amp, re, vr);
        vi = fma(pl.amp, im, vi);
    }
}

template <typename T, bool WRITE_VIS, bool DO_CHI2>
__global__ void __launch_bounds__(256) sample_multi_kernel(const SampleParams<T> p, const PlacementSet ps) {
    pdl_wait();
    const bool single = layout_single(p.ext, p.N);
    // a bound uv set (gal_plan_bind_uv): every cell is verified against the extent the transform was pruned to
    int ck_kumax = p.N, ck_rmin = 0, ck_rmax = p.N;
    if (p.ext_check) { ck_kumax = __ldcg(p.ext_check); ck_rmin = __ldcg(p.ext_check + 1); ck_rmax = __ldcg(p.ext_check + 2); }
    double acc = 0.0;
    unsigned int oob = 0, viol = 0;
    cx<T>* vis = reinterpret_cast<cx<T>*>(p.vis);
    for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k < p.M; k += (long long)gridDim.x * blockDim.x) {
        const double u = (double)__ldcs(p.u + k), v = (double)__ldcs(p.v + k);
        double vr = 0.0, vi = 0.0;
        if (ps.init_from_vis) { const cx<T> old = vis[k]; vr = (double)old.x; vi = (double)old.y; }
        if (single) multi_point<T, false>(p, ps, p.spec, u, v, vr, vi, oob, ck_kumax, ck_rmin, ck_rmax, viol);
        else multi_point<T, true>(p, ps, p.spec, u, v, vr, vi, oob, ck_kumax, ck_rmin, ck_rmax, viol);
        if (WRITE_VIS) vis[k] = mk<T>((T)vr, (T)vi);
        if (DO_CHI2) {                                                        // PAPER.md:718 (Eq. 10)
            const double dr = vr - (double)__ldcs(p.re_obs + k), di = vi - (double)__ldcs(p.im_obs + k);
            acc = fma(fma(dr, dr, di * di), (double)__ldcs(p.w + k), acc);
        }
    }
    sample_finish<T, DO_CHI2>(p, 0, acc, oob, viol);
}

// Extent of a point set under ANY rotation, from its largest baseline length (uv_radius_kernel): the index of a
// rotated coordinate is at most r_max / du, two cells of margin for the rounding of the listing's arithmetic;
// rows are symmetric about N/2.  One thread.
static __global__ void extent_from_radius_kernel(const unsigned long long* __restrict__ r2max_bits, double du, int N, int* ext) {
    pdl_wait();
    const double imax = sqrt(__longlong_as_double((long long)*r2max_bits)) * (1.0 + 1e-12) / du;
    const int H = N / 2;
    int e0 = H, e1 = 0, e2 = N - 1;
    if (imax + 3.0 < (double)(H - 1)) {
        const int k = (int)imax + 2;
        e0 = k + 1; e1 = H - k - 1; e2 = H + k + 1;
    }
    ext[0] = e0; ext[1] = e1; ext[2] = e2;
}

// total of a chunked batch: chi2_total = sum of the per-channel values in channel order (reading A17); one thread
static __global__ void sum_channels_kernel(const double* __restrict__ chi2_pc, int C, double* __restrict__ chi2_tot) {
    pdl_wait();
    double t = 0.0;
    for (int i = 0; i < C; ++i) t += chi2_pc[i];
    *chi2_tot = t;
}

// max over the points of u^2 + v^2 (bit pattern of a non-negative double orders like an integer): the
// rotation-invariant bound a bound uv set's extent is derived from (gal_plan_bind_uv).
template <typename T>
__global__ void __launch_bounds__(256) uv_radius_kernel(const T* __restrict__ u, const T* __restrict__ v, long long total,
                                                        unsigned long long* r2max_bits) {
    double m = 0.0;
    for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k < total; k += (long long)gridDim.x * blockDim.x) {
        const double a = (double)__ldcs(u + k), b = (double)__ldcs(v + k);
        const double r2 = fma(a, a, b * b);
        // fmax drops a NaN operand: a NaN coordinate counts as an infinite baseline, which the bind call rejects
        m = (r2 == r2) ? fmax(m, r2) : __longlong_as_double(0x7ff0000000000000LL);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
    if ((threadIdx.x & 31) == 0) atomicMax(r2max_bits, (unsigned long long)__double_as_longlong(m));
}

}  // namespace galb
