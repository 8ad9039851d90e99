// fft.cuh — hand-written 2-D real-to-complex FFT for sm_100a (no cuFFT).
//
// Computes F = rfft2(fftshift(image)) followed by fftshift along axis 0,
// stored u-major as column pairs: pair[b][ku][kvs] = {F[ku][kvs], F[ku+1][kvs]}, ku = 0..N/2,
// kvs = (kv + N/2) mod N — every value is stored twice (as .a of its own column and .b of the
// column before), so the four nodes of an interpolation cell are two adjacent, sector-aligned
// entries (64 contiguous bytes in fp64): exactly two 32-byte L2 sectors per sampled point instead
// of three, and one 128-byte line instead of two (sample.cuh).  The row pass writes its
// intermediate (the row-transformed image, transposed) to a separate u-major array work[b][ku][i].
//   * S2 (centre shift of the image) is never a pass: for even N it equals multiplying the
//     spectrum by (-1)^(ku+kv), applied in the last store of the column pass.
//   * S4 (shift along v) is an index fold in that same store.
//   * Row pass: one real row of N samples is read as N/2 complex numbers z[n] = x[2n] + i x[2n+1],
//     transformed with an (N/2)-point complex FFT in shared memory and untangled into the N/2+1
//     half-spectrum values; F rows per CTA are written TRANSPOSED (F*16 B contiguous per ku) so the
//     column pass reads and writes contiguous 16*N-byte columns.  L2 merges the partial lines.
//   * Column pass: work -> pair, one column per FFT, three radix passes through shared memory.
//   * With SWEEP the row loader evaluates the swept profile instead of reading an
//     image, so *Profile calls never materialise the image.
//
// The 1-D FFT of length L = R1*R2*R3 is a three-step Cooley-Tukey decomposition, all steps in
// registers with radix-R butterflies, exchanging through a padded shared-memory cube:
//   n = R2R3*n1 + R3*a + b,   k = k1 + R1*(c + R2*d)
//   step 1: DFT_R1 over n1, twiddle W_L^(n2*k1)           (n2 = R3*a + b)
//   step 2: DFT_R2 over a,  twiddle W_(R2R3)^(b*c)        (in place per work item)
//   step 3: DFT_R3 over b                                 (in place, or straight to global memory)
// Shared-memory address of element (k1, a|c, b|d): k1*P1 + (a|c)*R3 + (b|d), P1 = R2*R3 + 1 (odd),
// which makes every access pattern of the three steps bank-conflict free for 8/16-byte elements.
#pragma once
#include "common.cuh"

namespace galb {

// ------------------------------------------------------------------------------------------
// Radix-R DFTs on register arrays, forward kernel exp(-2 pi i nk/R), natural-order output.
// ------------------------------------------------------------------------------------------
template <typename T, int R> struct Dft;

template <typename T> struct Dft<T, 1> { static __device__ __forceinline__ void run(cx<T>*) {} };

template <typename T> struct Dft<T, 2> {
    static __device__ __forceinline__ void run(cx<T>* a) {
        cx<T> t = a[0];
        a[0] = cadd(t, a[1]);
        a[1] = csub(t, a[1]);
    }
};

template <typename T> struct Dft<T, 4> {
    static __device__ __forceinline__ void run(cx<T>* a) {
        cx<T> s02 = cadd(a[0], a[2]), d02 = csub(a[0], a[2]);
        cx<T> s13 = cadd(a[1], a[3]), d13 = mul_mi(csub(a[1], a[3]));
        a[0] = cadd(s02, s13);
        a[2] = csub(s02, s13);
        a[1] = cadd(d02, d13);
        a[3] = csub(d02, d13);
    }
};

template <typename T> struct Dft<T, 8> {
    static __device__ __forceinline__ void run(cx<T>* a) {
        const T h = (T)0.70710678118654752440;
        cx<T> e[4] = {a[0], a[2], a[4], a[6]};
        cx<T> o[4] = {a[1], a[3], a[5], a[7]};
        Dft<T, 4>::run(e);
        Dft<T, 4>::run(o);
        // o[k] *= exp(-2 pi i k / 8)
        o[1] = mk<T>((o[1].x + o[1].y) * h, (o[1].y - o[1].x) * h);
        o[2] = mul_mi(o[2]);
        o[3] = mk<T>((o[3].y - o[3].x) * h, -(o[3].x + o[3].y) * h);
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            a[k] = cadd(e[k], o[k]);
            a[k + 4] = csub(e[k], o[k]);
        }
    }
};

template <typename T> struct Dft<T, 16> {
    static __device__ __forceinline__ void run(cx<T>* a) {
        const T h = (T)0.70710678118654752440;
        const T c1 = (T)0.92387953251128675613;  // cos(pi/8)
        const T s1 = (T)0.38268343236508977173;  // sin(pi/8)
        cx<T> e[8], o[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) { e[k] = a[2 * k]; o[k] = a[2 * k + 1]; }
        Dft<T, 8>::run(e);
        Dft<T, 8>::run(o);
        // o[k] *= exp(-2 pi i k / 16) = (cos(pi k/8), -sin(pi k/8))
        o[1] = cmul(o[1], mk<T>(c1, -s1));
        o[2] = mk<T>((o[2].x + o[2].y) * h, (o[2].y - o[2].x) * h);
        o[3] = cmul(o[3], mk<T>(s1, -c1));
        o[4] = mul_mi(o[4]);
        o[5] = cmul(o[5], mk<T>(-s1, -c1));
        o[6] = mk<T>((o[6].y - o[6].x) * h, -(o[6].x + o[6].y) * h);
        o[7] = cmul(o[7], mk<T>(-c1, -s1));
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            a[k] = cadd(e[k], o[k]);
            a[k + 8] = csub(e[k], o[k]);
        }
    }
};

// w[k] = w1^k for k = 1..R-1 from one table value, by a product tree of depth <= log2(R)
// (w[2j] = w[j]^2, w[2j+1] = w[j] w[j+1]): at most four roundings deep for R = 16.
template <typename T, int R>
__device__ __forceinline__ void twiddle_powers(cx<T> w1, cx<T>* w) {
    w[0] = mk<T>(1, 0);
    if (R > 1) w[1] = w1;
#pragma unroll
    for (int k = 2; k < R; ++k) w[k] = (k & 1) ? cmul(w[k / 2], w[k / 2 + 1]) : cmul(w[k / 2], w[k / 2]);
}

// w * exp(-2 pi i d / M) for M = 8 or 16 and a compile-time d (after unrolling): the roots of unity are literals.
template <typename T, int M>
__device__ __forceinline__ cx<T> mul_root(cx<T> w, int d) {
    const T h = (T)0.70710678118654752440, c1 = (T)0.92387953251128675613, s1 = (T)0.38268343236508977173;
    const int e = (M == 16) ? d : 2 * d;                          // exponent in 16ths of a turn
    switch (e & 15) {
        case 0: return w;
        case 1: return cmul(w, mk<T>(c1, -s1));
        case 2: return mk<T>((w.x + w.y) * h, (w.y - w.x) * h);
        case 3: return cmul(w, mk<T>(s1, -c1));
        case 4: return mul_mi(w);
        case 5: return cmul(w, mk<T>(-s1, -c1));
        case 6: return mk<T>((w.y - w.x) * h, -(w.x + w.y) * h);
        case 7: return cmul(w, mk<T>(-c1, -s1));
        case 8: return mk<T>(-w.x, -w.y);
        case 9: return cmul(w, mk<T>(-c1, s1));
        case 10: return mk<T>(-(w.x + w.y) * h, (w.x - w.y) * h);
        case 11: return cmul(w, mk<T>(-s1, c1));
        case 12: return mk<T>(-w.y, w.x);
        case 13: return cmul(w, mk<T>(s1, c1));
        case 14: return mk<T>((w.x - w.y) * h, (w.x + w.y) * h);
        default: return cmul(w, mk<T>(c1, s1));
    }
}

// ------------------------------------------------------------------------------------------
// Geometry of one L-point FFT in shared memory.
// ------------------------------------------------------------------------------------------
constexpr int cmax(int a, int b) { return a > b ? a : b; }

template <typename T, int R1, int R2, int R3, int F> struct Geom {
    static constexpr int L = R1 * R2 * R3;
    static constexpr int RMAX = cmax(R1, cmax(R2, R3));
    static constexpr int TPF = L / RMAX;                                // threads per FFT
    static constexpr int NT = TPF * F;                                  // threads per CTA
    static constexpr int P1 = (R2 * R3 > 1) ? R2 * R3 + 1 : 1;          // k1 stride (odd)
    static constexpr int BG = 128 / (int)sizeof(cx<T>);                 // elements per 128 B of banks
    static constexpr int SKEW = (F >= BG) ? 1 : BG / F;                 // region stride mod BG
    static constexpr int BASE = R1 * P1;
    static constexpr int REGION = BASE + ((SKEW - BASE % BG) % BG + BG) % BG;
    static constexpr size_t SMEM = (size_t)REGION * F * sizeof(cx<T>);
    static __device__ __forceinline__ int zaddr(int k) {                // where X[k] sits after step 3
        return (k % R1) * P1 + ((k / R1) % R2) * R3 + k / (R1 * R2);
    }
};

// Steps 1 and 2.  S = this FFT's shared-memory region, t = thread index inside the FFT,
// tw[m * tws] = exp(-2 pi i m / L), load(n) returns input element n.  Ends with a barrier.
template <typename T, int R1, int R2, int R3, int TPF, typename LoadFn>
__device__ __forceinline__ void fft_steps12(cx<T>* S, int t, const cx<T>* __restrict__ tw, int tws, LoadFn load) {
    constexpr int P1 = (R2 * R3 > 1) ? R2 * R3 + 1 : 1;
    constexpr int N2 = R2 * R3;
    // The only table reads: one base twiddle per work item and step, W_L^n2 and W_(R2R3)^b.  They are
    // issued before the data loads so their latency hides behind them; the powers are formed in registers.
    cx<T> wb1 = mk<T>(1, 0), wb2 = mk<T>(1, 0);
    if (N2 > 1) wb1 = __ldg(tw + t * tws);
    if (R2 > 1 && R3 > 1) wb2 = __ldg(tw + (t % R3) * (R1 * tws));
    for (int n2 = t; n2 < N2; n2 += TPF) {
        cx<T> a[R1];
#pragma unroll
        for (int n1 = 0; n1 < R1; ++n1) a[n1] = load(N2 * n1 + n2);
        if (N2 > 1 && n2 != t) wb1 = __ldg(tw + n2 * tws);
        Dft<T, R1>::run(a);
        S[n2] = a[0];
        if (N2 > 1) {
            cx<T> w[R1];
            twiddle_powers<T, R1>(wb1, w);
#pragma unroll
            for (int k1 = 1; k1 < R1; ++k1) S[k1 * P1 + n2] = cmul(a[k1], w[k1]);
        } else {
#pragma unroll
            for (int k1 = 1; k1 < R1; ++k1) S[k1 * P1 + n2] = a[k1];
        }
    }
    __syncthreads();
    if (R2 > 1) {
        for (int it = t; it < R1 * R3; it += TPF) {
            const int b = it % R3, k1 = it / R3;
            cx<T>* base = S + k1 * P1 + b;
            cx<T> a[R2];
#pragma unroll
            for (int i = 0; i < R2; ++i) a[i] = base[i * R3];
            if (R3 > 1 && (TPF % R3) != 0 && it != t) wb2 = __ldg(tw + b * (R1 * tws));
            Dft<T, R2>::run(a);
            base[0] = a[0];
            if (R3 > 1) {
                cx<T> w[R2];
                twiddle_powers<T, R2>(wb2, w);
#pragma unroll
                for (int c = 1; c < R2; ++c) base[c * R3] = cmul(a[c], w[c]);
            } else {
#pragma unroll
                for (int c = 1; c < R2; ++c) base[c * R3] = a[c];
            }
        }
        __syncthreads();
    }
}

// ------------------------------------------------------------------------------------------
// Sweep: pixel value of the swept profile, every operation in the order of the
// listing and individually rounded (no FMA contraction) so that the hard-edge decisions
// r < Rmin, r > Rmax agree with a plain IEEE evaluation.
// ------------------------------------------------------------------------------------------
// a / b, correctly rounded, from r = RN(1 / b) (Markstein; see sample.cuh div_by): bit-identical to the IEEE
// division the listing performs, at 3 FP64 operations instead of a division sequence.
__device__ __forceinline__ double div_exact(double a, double b, double r, int true_div) {
    if (true_div) return __ddiv_rn(a, b);
    const double q0 = __dmul_rn(a, r);
    return __fma_rn(__fma_rn(-q0, b, a), r, q0);
}
// (double)n for 0 <= n < 2^31 without the conversion pipe: 2^52 + n is exact, minus 2^52
__device__ __forceinline__ double int_to_double(int n) {
    return __dsub_rn(__hiloint2double(0x43300000, n), 4503599627370496.0);
}

template <typename T>
__device__ __forceinline__ double sweep_pixel(const SweepParams& sp, int N, int i, int j) {
    // N is a power of two: i / N is the exact product i * (1 / N).  The other divisions use the reciprocal
    // shortcut; floor() and the int <-> double conversions go through the 2^52 mantissa trick (all exact).
    const double fN = int_to_double(N), rN = 1.0 / fN;
    const double y = __dmul_rn(__dmul_rn(__dsub_rn(0.5, __dmul_rn(int_to_double(i), rN)), sp.dxy), fN);
    const double x = __dmul_rn(__dmul_rn(__dsub_rn(0.5, __dmul_rn(int_to_double(j), rN)), sp.dxy), fN);
    const double xs = div_exact(x, sp.inc_cos, sp.r_inc, sp.true_div);
    const double r = __dsqrt_rn(__dadd_rn(__dmul_rn(xs, xs), __dmul_rn(y, y)));
    if (!(r >= sp.Rmin && r <= sp.Rmax)) return 0.0;
    const double pos = div_exact(__dsub_rn(r, sp.Rmin), sp.dR, sp.r_dR, sp.true_div);
    // k = floor(pos) clamped to [0, nr - 2]; pos >= 0 here and far below 2^31 (pos <= nr - 1 + rounding)
    const double tk = __dadd_rn(pos, 4503599627370496.0);
    int k = __double2loint(tk);
    if (__dsub_rn(tk, 4503599627370496.0) > pos) k -= 1;
    if (k >= sp.nr - 1) k = sp.nr - 2;
    if (k < 0) k = 0;
    const double t = __dsub_rn(pos, int_to_double(k));
    const T* I = (const T*)sp.I;
    const double i0 = (double)__ldg(I + k), i1 = (double)__ldg(I + k + 1);
    const double val = __dadd_rn(i0, __dmul_rn(t, __dsub_rn(i1, i0)));
    return __dmul_rn(__dmul_rn(val, sp.dxy), sp.dxy);
}

// ------------------------------------------------------------------------------------------
// Row pass.
// ------------------------------------------------------------------------------------------
template <typename T> struct RowParams {
    const T* image;        // [rows_total][N] (unused with SWEEP)
    cx<T>* spec;           // work[batch][N/2+1][N]: the row-transformed image, transposed
    const cx<T>* tw;       // exp(-2 pi i m / N), m = 0..N-1
    int N;
    int rows_total;        // batch * N
    const int* ext;        // {largest column ku needed, first row kvs, last row kvs} (sample.cuh, uv extent)
    int pf_blocks;         // > 0: CTA b asks the L2 for the image rows of CTA b + pf_blocks (the CTAs resident at once)
    SweepParams sweep;
};

// CTA `blk` of a grid of row blocks (rows_per_block rows each) prefetches the rows of block blk + pf_blocks into the
// L2.  The image is an input of the call, not a product of the kernel before in the chain, so this runs before the
// programmatic dependency is waited for.
template <typename T>
__device__ __forceinline__ void prefetch_row_block(const RowParams<T>& p, long long blk, int rows_per_block) {
    if (p.pf_blocks <= 0 || threadIdx.x >= rows_per_block) return;
    const long long row = (blk + p.pf_blocks) * rows_per_block + threadIdx.x;
    if (row < p.rows_total) l2_prefetch_bulk(p.image + row * (long long)p.N, (uint32_t)(p.N * sizeof(T)));
}

// One block of F image rows (block index vb): transform, untangle, transposed write.  Shared by the row-pass kernel
// (one block per CTA) and the conditional second pass of a call (redo_kernel).
template <typename T, int R1, int R2, int R3, int F, bool SWEEP>
__device__ __forceinline__ void row_block(const RowParams<T>& p, const long long vb, cx<T>* smem) {
    using G = Geom<T, R1, R2, R3, F>;
    constexpr int L = G::L;                    // = N / 2
    const int tid = threadIdx.x;
    const int f = tid / G::TPF, t = tid % G::TPF;
    const int N = p.N;
    const long long row0 = vb * F;
    const long long row = row0 + f;
    const bool valid = row < p.rows_total;
    cx<T>* S = smem + f * G::REGION;

    if (SWEEP) {
        const int i = (int)(row % N);
        fft_steps12<T, R1, R2, R3, G::TPF>(S, t, p.tw, 2, [&](int n) -> cx<T> {
            if (!valid) return mk<T>(0, 0);
            return mk<T>((T)sweep_pixel<T>(p.sweep, N, i, 2 * n), (T)sweep_pixel<T>(p.sweep, N, i, 2 * n + 1));
        });
    } else {
        const cx<T>* z = reinterpret_cast<const cx<T>*>(p.image + (valid ? row : 0) * (long long)N);
        fft_steps12<T, R1, R2, R3, G::TPF>(S, t, p.tw, 2, [&](int n) -> cx<T> {
            return valid ? __ldcs(z + n) : mk<T>(0, 0);
        });
    }
    // step 3, in place: X[k1 + R1*(c + R2*d)] -> S[k1*P1 + c*R3 + d]
    if (R3 > 1) {
        for (int it = t; it < R1 * R2; it += G::TPF) {
            const int k1 = it % R1, c = it / R1;
            cx<T>* base = S + k1 * G::P1 + c * R3;
            cx<T> a[R3];
#pragma unroll
            for (int b = 0; b < R3; ++b) a[b] = base[b];
            Dft<T, R3>::run(a);
#pragma unroll
            for (int d = 0; d < R3; ++d) base[d] = a[d];
        }
        __syncthreads();
    }
    // Untangle the packed real FFT and write F rows transposed.
    //   E = (Z[k] + conj Z[L-k]) / 2,  O = -i (Z[k] - conj Z[L-k]) / 2,  W = exp(-2 pi i k / N)
    //   X[k] = E + W O,   X[L-k] = conj(E - W O)     (k = 0 gives X[0] and X[L])
    const int NU = N / 2 + 1;
    const long long b_img = row0 / N;
    const int i0 = (int)(row0 % N);
    cx<T>* out = p.spec + b_img * (long long)NU * N + i0;
    const int rows_here = (int)((p.rows_total - row0) < F ? (p.rows_total - row0) : F);
    // columns beyond the uv extent are never sampled: neither formed nor written
    const int kumax = __ldcg(p.ext);
    const int kend = kumax < L / 2 ? kumax : L / 2;
    for (int idx = tid; idx < F * (kend + 1); idx += G::NT) {
        const int ff = idx % F, k = idx / F;
        if (ff >= rows_here) continue;
        const cx<T>* Sf = smem + ff * G::REGION;
        const cx<T> zk = Sf[G::zaddr(k)];
        const cx<T> zm = Sf[G::zaddr((L - k) % L)];
        const cx<T> E = mk<T>(zk.x + zm.x, zk.y - zm.y);          // 2 E and 2 O: the factor 1/2 is folded into
        const cx<T> O = mk<T>(zk.y + zm.y, zm.x - zk.x);          // the column pass's sign (exact)
        const cx<T> WO = cmul(__ldg(p.tw + k), O);
        const cx<T> xk = cadd(E, WO);
        cx<T> xm = csub(E, WO);
        xm.y = -xm.y;
        out[(long long)k * N + ff] = xk;
        if (L - k <= kumax) out[(long long)(L - k) * N + ff] = xm;
    }
}

template <typename T, int R1, int R2, int R3, int F, bool SWEEP>
__global__ void __launch_bounds__(Geom<T, R1, R2, R3, F>::NT)
row_pass_kernel(const RowParams<T> p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    if (!SWEEP) prefetch_row_block(p, blockIdx.x, F);
    pdl_wait();
    row_block<T, R1, R2, R3, F, SWEEP>(p, blockIdx.x, reinterpret_cast<cx<T>*>(smem_raw));
}

// ------------------------------------------------------------------------------------------
// Row pass, pipelined (nxy = 1024 .. 4096; same result as row_pass_kernel).
//
// Persistent CTAs (one per SM).  A CTA is NG groups of GT = TPF * F consumer threads plus one producer warp.
// A group transforms F adjacent image rows at a time, LANE-INTERLEAVED: thread gtid works on row gtid % F as
// FFT thread gtid / F, so the F results for one ku sit in adjacent lanes and every store instruction writes
// F * sizeof(complex) contiguous bytes per ku (whole 32-byte sectors in fp64 with F = 2).
//   * Staging: lane 0 of the producer warp streams whole rows with `cp.async.bulk` (TMA) into a ring of NS
//     slots (one slot = F row regions), full/empty mbarriers; the rows land linearly at the start of the
//     regions they are transformed in, so the loads of the next NS - NG row blocks are in flight while the
//     groups compute.  The image is an input of the call, not a product of the kernel before in the chain, so
//     the producer does not wait for the programmatic dependency: its first loads overlap the kernel before.
//   * Step 1 reads the linear row (conflict free), a group barrier separates those reads from the writes of
//     the padded cube; step 2 is in place; step 3 is FUSED with the real-FFT untangle in registers: a thread
//     takes a work item (k1, c) together with the item that holds the mirrored indices L - k —
//     (R1 - k1, R2 - 1 - c) for k1 != 0, (0, R2 - c) for k1 = 0 — so Z[k] and Z[L - k] of all its outputs are
//     its own registers: no third exchange through shared memory, no barrier, and the slot is released to
//     the producer as soon as the step-3 operands are read.
//   * Groups synchronise with named barriers (bar.sync id, GT), never the whole CTA, so the NG groups drift
//     into different phases and the FP64 pipe, the shared-memory pipe and the store path overlap.
// ------------------------------------------------------------------------------------------
template <typename T, int R1, int R2, int R3, int F> struct RowGeom {
    static constexpr int L = R1 * R2 * R3;
    static constexpr int RMAX = cmax(R1, cmax(R2, R3));
    static_assert(R1 == RMAX, "step 1 must be exactly one work item per thread (in-place landing buffer)");
    static_assert(R2 >= 2 && R3 >= 2 && R1 % 2 == 0 && R2 % 2 == 0 && R3 % 2 == 0, "three-step plans only");
    static constexpr int TPF = L / RMAX;                                // threads per row
    static constexpr int GT = TPF * F;                                  // threads per group
    static_assert(GT % 32 == 0, "a group is a whole number of warps");
    static constexpr int P1 = R2 * R3 + 1;
    static constexpr int BG = 128 / (int)sizeof(cx<T>);
    static_assert(F <= BG, "rows per group");
    static constexpr int SKEW = BG / F;                                 // region stride mod BG: rows interleave the banks
    static constexpr int BASE = R1 * P1;                                // >= L: the linear row fits
    static constexpr int REGION = BASE + ((SKEW - BASE % BG) % BG + BG) % BG;
    static constexpr uint32_t SLOT_BYTES = (uint32_t)REGION * F * sizeof(cx<T>);
    static_assert((REGION * sizeof(cx<T>)) % 16 == 0, "bulk-copy destination alignment");
};

__device__ __forceinline__ void group_barrier(int id, int nthreads) {
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}
__device__ __forceinline__ void fence_proxy_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// Where step 1 takes its input from: the TMA ring (persistent CTAs, one per SM), plain global loads (one row block
// per CTA, several CTAs per SM: no producer warp, no ring), or the swept profile.
enum RowLoad { ROW_TMA = 0, ROW_DIRECT = 1, ROW_SWEEP = 2 };
#ifndef GAL_ROW_F1_MINB
#define GAL_ROW_F1_MINB 4            // resident CTAs per SM the one-row-per-CTA form (128 threads) is compiled for
#endif

template <typename T, int R1, int R2, int R3, int F, int NG, int NS, int MODE>
__global__ void __launch_bounds__(RowGeom<T, R1, R2, R3, F>::GT * NG + (MODE == ROW_TMA ? 32 : 0),
                                  MODE == ROW_TMA ? 1 : (RowGeom<T, R1, R2, R3, F>::GT * NG == 128 ? GAL_ROW_F1_MINB : cmax(2, 512 / (RowGeom<T, R1, R2, R3, F>::GT * NG))))
row_pipe_kernel(const RowParams<T> p) {
    constexpr bool SWEEP = MODE != ROW_TMA;          // "no ring": inputs do not come through the mbarrier pipeline
    using G = RowGeom<T, R1, R2, R3, F>;
    constexpr int L = G::L, TPF = G::TPF, GT = G::GT, P1 = G::P1, REGION = G::REGION;
    constexpr int N2 = R2 * R3, H1 = R1 / 2, NPAIR = R1 * R2 / 2;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    cx<T>* smem = reinterpret_cast<cx<T>*>(smem_raw);
    const uint32_t full0 = smem_u32(smem_raw) + NS * G::SLOT_BYTES, empty0 = full0 + 8 * NS;
    const int tid = threadIdx.x, lane = tid & 31;
    const int N = p.N;
    const long long nblk = p.rows_total / F;                 // F divides nxy: a block never straddles two images
    if (MODE == ROW_TMA) {
        if (tid == 0) {
            for (int s = 0; s < NS; ++s) { mbar_init(full0 + 8 * s, 1); mbar_init(empty0 + 8 * s, GT / 32); }
            mbar_fence_init();
        }
        __syncthreads();
    }

    if (MODE == ROW_TMA && tid >= NG * GT) {                 // ---- producer warp ----
        if (lane == 0) {
            const uint64_t pol = l2_policy_evict_first();
            const uint32_t row_bytes = (uint32_t)N * sizeof(T);
            uint32_t slot = 0, parity = 1;                   // a fresh mbarrier lets a wait on parity 1 through
            for (long long blk = blockIdx.x; blk < nblk; blk += gridDim.x) {
                mbar_wait_relaxed(empty0 + 8 * slot, parity);
                const uint32_t mb = full0 + 8 * slot;
                const uint32_t dst = smem_u32(smem_raw) + slot * G::SLOT_BYTES;
                mbar_expect_tx(mb, F * row_bytes);
#pragma unroll
                for (int f = 0; f < F; ++f)
                    tma_load_1d(dst + f * (uint32_t)(REGION * sizeof(cx<T>)), p.image + (blk * F + f) * (long long)N, row_bytes, mb, pol);
                if (++slot == NS) { slot = 0; parity ^= 1u; }
            }
        }
        return;
    }

    // ---- consumer groups ----
    const int g = tid / GT, gtid = tid % GT;
    const int t = gtid / F, f = gtid % F;
    const int bar_id = 1 + g;
    if (MODE == ROW_DIRECT) prefetch_row_block(p, blockIdx.x, F);
    pdl_wait();
    const int kumax = __ldcg(p.ext);
    const int NU = N / 2 + 1;
    const cx<T>* __restrict__ tw = p.tw;
    // the only table reads of steps 1 and 2: one base twiddle each, W_L^t and W_(R2 R3)^(t mod R3)
    const cx<T> wb1 = __ldg(tw + 2 * t);
    static_assert(TPF % R3 == 0, "the step-2 twiddle index is the same for every work item of a thread");
    const cx<T> wb2 = __ldg(tw + (t % R3) * (2 * R1));
    long long q = g;
    for (long long blk = blockIdx.x + (long long)gridDim.x * g; blk < nblk; blk += (long long)gridDim.x * NG, q += NG) {
        const int slot = SWEEP ? g : (int)(q % NS);           // (no ring without the producer: one slot per group)
        const uint32_t par = (uint32_t)((q / NS) & 1);
        cx<T>* S = smem + (size_t)slot * F * REGION + (size_t)f * REGION;
        const long long row = blk * F + f;
        // step 1: DFT_R1 over n1, twiddle W_L^(n2 k1), n2 = t
        {
            cx<T> a[R1];
            if (MODE == ROW_SWEEP) {
                const int i = (int)(row % N);
#pragma unroll
                for (int n1 = 0; n1 < R1; ++n1) {
                    const int n = N2 * n1 + t;
                    a[n1] = mk<T>((T)sweep_pixel<T>(p.sweep, N, i, 2 * n), (T)sweep_pixel<T>(p.sweep, N, i, 2 * n + 1));
                }
            } else if (MODE == ROW_DIRECT) {
                const cx<T>* z = reinterpret_cast<const cx<T>*>(p.image + row * (long long)N);
#pragma unroll
                for (int n1 = 0; n1 < R1; ++n1) a[n1] = __ldcs(z + N2 * n1 + t);
            } else {
                mbar_wait(full0 + 8 * slot, par);
#pragma unroll
                for (int n1 = 0; n1 < R1; ++n1) a[n1] = S[N2 * n1 + t];
                group_barrier(bar_id, GT);                   // every linear read before the first padded write
            }
            Dft<T, R1>::run(a);
            S[t] = a[0];
            cx<T> w[R1];
            twiddle_powers<T, R1>(wb1, w);
#pragma unroll
            for (int k1 = 1; k1 < R1; ++k1) S[k1 * P1 + t] = cmul(a[k1], w[k1]);
        }
        group_barrier(bar_id, GT);
        // step 2: DFT_R2 over a, twiddle W_(R2 R3)^(b c), in place per work item
        for (int it = t; it < R1 * R3; it += TPF) {
            const int b = it % R3, k1 = it / R3;
            cx<T>* base = S + k1 * P1 + b;
            cx<T> a[R2];
#pragma unroll
            for (int i = 0; i < R2; ++i) a[i] = base[i * R3];
            Dft<T, R2>::run(a);
            base[0] = a[0];
            cx<T> w[R2];
            twiddle_powers<T, R2>(wb2, w);
#pragma unroll
            for (int c = 1; c < R2; ++c) base[c * R3] = cmul(a[c], w[c]);
        }
        group_barrier(bar_id, GT);
        // step 3 fused with the untangle of the packed real transform:
        //   E = (Z[k] + conj Z[L-k]) / 2,  O = -i (Z[k] - conj Z[L-k]) / 2,  W = exp(-2 pi i k / N)
        //   X[k] = E + W O,   X[L-k] = conj(E - W O)     (k = 0 gives X[0] and X[L])
        cx<T>* out = p.spec + (row / N) * (long long)NU * N + (row % N);
        auto butterfly = [&](const cx<T> zk, const cx<T> zm, const cx<T> W, const int k) {
            const int km = L - k;
            const bool sk = k <= kumax, sm = km <= kumax;
            if (!sk && !sm) return;
            const cx<T> E = mk<T>(zk.x + zm.x, zk.y - zm.y);      // 2 E and 2 O: the factor 1/2 is folded into the
            const cx<T> O = mk<T>(zk.y + zm.y, zm.x - zk.x);      // column pass's sign (exact)
            const cx<T> WO = cmul(W, O);
            if (sk) out[(long long)k * N] = cadd(E, WO);
            if (sm) { cx<T> xm = csub(E, WO); xm.y = -xm.y; out[(long long)km * N] = xm; }
        };
        bool released = SWEEP;
        for (int j = t; j < NPAIR; j += TPF) {
            const int k1h = j % H1, cc = j / H1;
            int pk1, pc, qk1, qc;
            bool special = false;
            if (k1h != 0) { pk1 = k1h; pc = cc; qk1 = R1 - k1h; qc = R2 - 1 - cc; }
            else if (cc < R2 / 2) { pk1 = H1; pc = cc; qk1 = H1; qc = R2 - 1 - cc; }
            else if (cc > R2 / 2) { pk1 = 0; pc = cc - R2 / 2; qk1 = 0; qc = R2 - pc; }
            else { special = true; pk1 = 0; pc = 0; qk1 = 0; qc = R2 / 2; }      // the two self-mirrored items
            // untangle twiddles W_N^k, k = k0 + R1 R2 d: one table value times the (2 R3)-th roots of unity, formed
            // in registers (with the ring resident the L1 is too small to keep the table)
            const cx<T> w0 = __ldg(tw + (pk1 + R1 * pc));
            const cx<T> w0b = special ? __ldg(tw + R1 * (R2 / 2)) : w0;
            cx<T> a[R3], m[R3];
            {
                const cx<T>* pa = S + pk1 * P1 + pc * R3;
                const cx<T>* pm = S + qk1 * P1 + qc * R3;
#pragma unroll
                for (int b = 0; b < R3; ++b) { a[b] = pa[b]; m[b] = pm[b]; }
            }
            if (!SWEEP && j + TPF >= NPAIR) {                // this thread's last read of the slot: hand it back
                fence_proxy_async_smem();
                __syncwarp();
                if (lane == 0) mbar_arrive(empty0 + 8 * slot);
                released = true;
            }
            Dft<T, R3>::run(a);
            Dft<T, R3>::run(m);
            if (!special) {
#pragma unroll
                for (int d = 0; d < R3; ++d)
                    butterfly(a[d], m[R3 - 1 - d], mul_root<T, 2 * R3>(w0, d), pk1 + R1 * (pc + R2 * d));
            } else {
                butterfly(a[0], a[0], mk<T>(1, 0), 0);
#pragma unroll
                for (int d = 1; d <= R3 / 2; ++d) butterfly(a[d], a[R3 - d], mul_root<T, 2 * R3>(mk<T>(1, 0), d), R1 * R2 * d);
#pragma unroll
                for (int d = 0; d < R3 / 2; ++d)
                    butterfly(m[d], m[R3 - 1 - d], mul_root<T, 2 * R3>(w0b, d), R1 * (R2 / 2 + R2 * d));
            }
        }
        if (!released) {                                     // warps without a step-3 work item (NPAIR < TPF)
            fence_proxy_async_smem();
            __syncwarp();
            if (lane == 0) mbar_arrive(empty0 + 8 * slot);
        }
        if (SWEEP) group_barrier(bar_id, GT);                // the region is rewritten by the next block's step 1
    }
}

// ------------------------------------------------------------------------------------------
// Column pass (in place).
// ------------------------------------------------------------------------------------------
// Layout of the sampled spectrum.  A call pruned to a part of the half plane writes COLUMN PAIRS
// (pair[ku][kvs] = {F[ku][kvs], F[ku+1][kvs]}, every value twice: two sectors per sampled point; the doubled
// write is a few MB).  A call that needs the WHOLE half plane (extent == {N/2, 0, N-1}: pruning off, or points
// that wrap, reading A6) writes every value ONCE, single[ku][kvs]: the column pass then moves 2 instead of 3
// spectrum volumes and the gather pays three sectors per point instead of two.  Both layouts live in the same
// plan buffer; the column pass and the sampler take the decision from the same device-resident extent.
__device__ __forceinline__ bool extent_is_whole_plane(const int* ext, int N) {
#ifdef GAL_FORCE_PAIR
    return false;
#else
    return __ldcg(ext) >= N / 2 && __ldcg(ext + 1) <= 0 && __ldcg(ext + 2) >= N - 1;
#endif
}

template <typename T> struct ColParams {
    const cx<T>* work;     // [batch][N/2+1][N], written by the row pass
    NodePair<T>* pair;     // [batch][N/2+1][N], the sampled spectrum
    const cx<T>* tw;
    int N;
    long long cols_total;  // batch * (N/2+1)
    const int* ext;        // as RowParams::ext
    int pf_groups;         // > 0: CTA b asks the L2 for the columns of CTA b + pf_groups (whole-plane transforms only)
};

// One group of F adjacent columns, g0 .. g0 + F - 1 of the u-major work array: transform, sign / row folds, write
// the sampled spectrum.  Shared by the column-pass kernel and the conditional second pass of a call (redo_kernel).
template <typename T, int R1, int R2, int R3, int F>
__device__ __forceinline__ void col_block(const ColParams<T>& p, const long long g0, cx<T>* smem) {
    using G = Geom<T, R1, R2, R3, F>;
    constexpr int L = G::L;                    // = N
    const int tid = threadIdx.x;
    const int f = tid / G::TPF, t = tid % G::TPF;
    const int NU = L / 2 + 1;
    // uv extent: columns beyond kumax are skipped, rows outside [rmin, rmax] are not written
    const int kumax = __ldcg(p.ext), rmin = __ldcg(p.ext + 1), rmax = __ldcg(p.ext + 2);
    const bool single = extent_is_whole_plane(p.ext, L);
    cx<T>* S = smem + f * G::REGION;
    {
        const long long g = g0 + f;
        const int ku = (int)(g % NU);
        {
            bool any = false;
#pragma unroll
            for (int ff = 0; ff < F; ++ff) {
                const long long gg = g0 + ff;
                any = any || (gg < p.cols_total && (int)(gg % NU) <= kumax);
            }
            if (!any) return;
        }
        const bool valid = g < p.cols_total && ku <= kumax;
        const cx<T>* col = p.work + (valid ? g : 0) * (long long)L;
        NodePair<T>* own = p.pair + (valid ? g : 0) * (long long)L;          // .a of this column's entries
        NodePair<T>* prev = own - (ku > 0 ? L : 0);                          // .b of the entries one column down
        cx<T>* sown = reinterpret_cast<cx<T>*>(p.pair) + (valid ? g : 0) * (long long)L;   // single-copy layout

        fft_steps12<T, R1, R2, R3, G::TPF>(S, t, p.tw, 1, [&](int n) -> cx<T> {
            return valid ? col[n] : mk<T>(0, 0);
        });
        // step 3; kv = k1 + R1*(c + R2*d); sign (-1)^(ku+kv) folds the image centre shift, row (kv + N/2) mod N
        // folds the shift along v.  Each value goes to its own entry (.a) and to the entry of the column
        // before (.b).
        if constexpr (F == 1) {
            // one column per CTA: straight from registers to global memory, two 16-byte stores per value
            for (int it = t; it < R1 * R2; it += G::TPF) {
                const int k1 = it % R1, c = it / R1;
                const cx<T>* base = S + k1 * G::P1 + c * R3;
                cx<T> a[R3];
#pragma unroll
                for (int b = 0; b < R3; ++b) a[b] = base[b];
                Dft<T, R3>::run(a);
                if (valid) {
#pragma unroll
                    for (int d = 0; d < R3; ++d) {
                        const int kv = k1 + R1 * (c + R2 * d);
                        const T sgn = ((ku + kv) & 1) ? (T)-0.5 : (T)0.5;
                        const int kvs = (kv + L / 2) & (L - 1);
                        if (kvs >= rmin && kvs <= rmax) {
                            const cx<T> val = mk<T>(sgn * a[d].x, sgn * a[d].y);
                            if (single) {
                                sown[kvs] = val;
                            } else {
                                own[kvs].a = val;
                                if (ku > 0) prev[kvs].b = val;
                            }
                        }
                    }
                }
            }
        } else {
            // several adjacent columns per CTA: the signed results go back to shared memory and are written
            // out as whole entries {F[ku], F[ku+1]} (one 32-byte store in fp64, a full sector) wherever both
            // columns are in this CTA; only the first column's .b of the entry before and the last column's .a
            // remain half-sector stores.
            for (int it = t; it < R1 * R2; it += G::TPF) {
                const int k1 = it % R1, c = it / R1;
                cx<T>* base = S + k1 * G::P1 + c * R3;
                cx<T> a[R3];
#pragma unroll
                for (int b = 0; b < R3; ++b) a[b] = base[b];
                Dft<T, R3>::run(a);
                const T sgn = ((ku + k1) & 1) ? (T)-0.5 : (T)0.5;     // R1 is even: kv and k1 have one parity
#pragma unroll
                for (int d = 0; d < R3; ++d) base[d] = mk<T>(sgn * a[d].x, sgn * a[d].y);
            }
            __syncthreads();
            for (int idx = tid; idx < F * L; idx += G::NT) {
                const int ff = idx / L, kvs = idx % L;
                const long long gg = g0 + ff;
                const int kuf = (int)(gg % NU);
                if (gg >= p.cols_total || kuf > kumax || kvs < rmin || kvs > rmax) continue;
                const int za = G::zaddr((kvs + L / 2) & (L - 1));
                const cx<T> x = smem[ff * G::REGION + za];
                if (single) { reinterpret_cast<cx<T>*>(p.pair)[gg * (long long)L + kvs] = x; continue; }
                NodePair<T>* e = p.pair + gg * (long long)L + kvs;
                if (ff + 1 < F && kuf < L / 2 && kuf + 1 <= kumax) {
                    NodePair<T> pr;
                    pr.a = x;
                    pr.b = smem[(ff + 1) * G::REGION + za];
                    store_pair(e, pr);
                } else {
                    e->a = x;
                }
                if (ff == 0 && kuf > 0) (e - L)->b = x;
            }
        }
    }
}

template <typename T, int R1, int R2, int R3, int F>
__global__ void __launch_bounds__(Geom<T, R1, R2, R3, F>::NT)
col_pass_kernel(const ColParams<T> p) {
    constexpr int L = Geom<T, R1, R2, R3, F>::L;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    pdl_wait();
    // whole plane: the row-transformed image comes back from HBM (a pruned one is still in the L2): ask the L2 for
    // the columns of the CTA that will take this one's place
    if (p.pf_groups > 0 && threadIdx.x < F && extent_is_whole_plane(p.ext, L)) {
        const long long gg = ((long long)blockIdx.x + p.pf_groups) * F + threadIdx.x;
        if (gg < p.cols_total) l2_prefetch_bulk(p.work + gg * (long long)L, (uint32_t)(L * sizeof(cx<T>)));
    }
    col_block<T, R1, R2, R3, F>(p, (long long)blockIdx.x * F, reinterpret_cast<cx<T>*>(smem_raw));   // one group of F columns per CTA
}

// ------------------------------------------------------------------------------------------
// Column pass for N = 2 L beyond the longest three-step transform (N = 8192): one column per CTA as two
// interleaved L-point transforms (even and odd samples, the two regions of an F = 2 geometry) and one
// radix-2 combination  X[k] = E[k] + W_N^k O[k],  X[k + L] = E[k] - W_N^k O[k]  that writes straight to the
// column pairs with the same sign / row folds and pruning as col_pass_kernel.
// ------------------------------------------------------------------------------------------
template <typename T, int R1, int R2, int R3>
__global__ void __launch_bounds__(Geom<T, R1, R2, R3, 2>::NT)
col_pass_x2_kernel(const ColParams<T> p) {
    using G = Geom<T, R1, R2, R3, 2>;
    constexpr int L = G::L;                    // = N / 2
    constexpr int N = 2 * L, NU = N / 2 + 1;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cx<T>* smem = reinterpret_cast<cx<T>*>(smem_raw);
    const int tid = threadIdx.x;
    const int f = tid / G::TPF, t = tid % G::TPF;
    pdl_wait();
    const int kumax = __ldcg(p.ext), rmin = __ldcg(p.ext + 1), rmax = __ldcg(p.ext + 2);
    const long long g = blockIdx.x;
    const int ku = (int)(g % NU);
    if (ku > kumax) return;
    const cx<T>* col = p.work + g * (long long)N;
    NodePair<T>* own = p.pair + g * (long long)N;
    NodePair<T>* prev = own - (ku > 0 ? N : 0);
    cx<T>* sown = reinterpret_cast<cx<T>*>(p.pair) + g * (long long)N;
    const bool single = extent_is_whole_plane(p.ext, N);
    cx<T>* S = smem + f * G::REGION;

    fft_steps12<T, R1, R2, R3, G::TPF>(S, t, p.tw, 2, [&](int n) -> cx<T> { return col[2 * n + f]; });
    if (R3 > 1) {                              // step 3, in place (as in the row pass)
        for (int it = t; it < R1 * R2; it += G::TPF) {
            const int k1 = it % R1, c = it / R1;
            cx<T>* base = S + k1 * G::P1 + c * R3;
            cx<T> a[R3];
#pragma unroll
            for (int b = 0; b < R3; ++b) a[b] = base[b];
            Dft<T, R3>::run(a);
#pragma unroll
            for (int d = 0; d < R3; ++d) base[d] = a[d];
        }
    }
    __syncthreads();
    const cx<T>* SE = smem;
    const cx<T>* SO = smem + G::REGION;
    for (int k = tid; k < L; k += G::NT) {
        const cx<T> E = SE[G::zaddr(k)];
        const cx<T> WO = cmul(__ldg(p.tw + k), SO[G::zaddr(k)]);
        const T sgn = ((ku + k) & 1) ? (T)-0.5 : (T)0.5;          // L is even: kv = k and k + L have one parity
        const cx<T> x0 = cadd(E, WO), x1 = csub(E, WO);
        const int kvs0 = k + L, kvs1 = k;                     // (kv + N/2) mod N for kv = k, k + L
        if (kvs0 >= rmin && kvs0 <= rmax) {
            const cx<T> val = mk<T>(sgn * x0.x, sgn * x0.y);
            if (single) { sown[kvs0] = val; } else { own[kvs0].a = val; if (ku > 0) prev[kvs0].b = val; }
        }
        if (kvs1 >= rmin && kvs1 <= rmax) {
            const cx<T> val = mk<T>(sgn * x1.x, sgn * x1.y);
            if (single) { sown[kvs1] = val; } else { own[kvs1].a = val; if (ku > 0) prev[kvs1].b = val; }
        }
    }
}

// ------------------------------------------------------------------------------------------
// nxy = 16384 (the paper's largest size).  A row is 8192 complex numbers (128 KB in fp64), a
// column 16384 (256 KB): neither fits the three-step transform in one CTA's shared memory.
//   * Row pass: one row per CTA as two interleaved 4096-point transforms (even / odd samples of the packed
//     sequence z, the two regions of an F = 2 geometry), one radix-2 combination in place, then the real-FFT
//     untangle.  It writes image row i to position (i mod 4) N/4 + i / 4 of the u-major work array, i.e. already
//     DECIMATED BY FOUR for the column transform.
//   * Column transform N = 4 x 4096 (four-step through global memory):  X[k2 + 4096 k1] =
//       sum_n1 W_4^(n1 k1) W_N^(n1 k2) Y_n1[k2],   Y_n1 = DFT_4096 of x[n1 + 4 n2] (a contiguous quarter column).
//     col_sub_kernel transforms one quarter column per CTA in place and applies W_N^(n1 k2); col_comb4_kernel
//     does the four-point combination and writes the spectrum with the same sign / row folds, layouts and
//     pruning as col_pass_kernel.  Two extra passes over the reachable columns, nothing else.
// ------------------------------------------------------------------------------------------
template <typename T, int R1, int R2, int R3, bool SWEEP>
__global__ void __launch_bounds__(Geom<T, R1, R2, R3, 2>::NT)
row_pass_x2_kernel(const RowParams<T> p) {
    using G = Geom<T, R1, R2, R3, 2>;
    constexpr int LH = G::L;                   // = N / 4: length of each interleaved transform
    constexpr int L = 2 * LH;                  // = N / 2: length of the packed complex row
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cx<T>* smem = reinterpret_cast<cx<T>*>(smem_raw);
    const int tid = threadIdx.x;
    const int f = tid / G::TPF, t = tid % G::TPF;
    const int N = p.N;
    const long long row = blockIdx.x;
    cx<T>* S = smem + f * G::REGION;
    if (!SWEEP) prefetch_row_block(p, blockIdx.x, 1);
    pdl_wait();
    if (SWEEP) {
        const int i = (int)(row % N);
        fft_steps12<T, R1, R2, R3, G::TPF>(S, t, p.tw, 4, [&](int m) -> cx<T> {
            const int n = 2 * m + f;
            return mk<T>((T)sweep_pixel<T>(p.sweep, N, i, 2 * n), (T)sweep_pixel<T>(p.sweep, N, i, 2 * n + 1));
        });
    } else {
        const cx<T>* z = reinterpret_cast<const cx<T>*>(p.image + row * (long long)N);
        fft_steps12<T, R1, R2, R3, G::TPF>(S, t, p.tw, 4, [&](int m) -> cx<T> { return __ldcs(z + 2 * m + f); });
    }
    if (R3 > 1) {                              // step 3, in place
        for (int it = t; it < R1 * R2; it += G::TPF) {
            const int k1 = it % R1, c = it / R1;
            cx<T>* base = S + k1 * G::P1 + c * R3;
            cx<T> a[R3];
#pragma unroll
            for (int b = 0; b < R3; ++b) a[b] = base[b];
            Dft<T, R3>::run(a);
#pragma unroll
            for (int d = 0; d < R3; ++d) base[d] = a[d];
        }
    }
    __syncthreads();
    cx<T>* SE = smem;
    cx<T>* SO = smem + G::REGION;
    for (int k = tid; k < LH; k += G::NT) {    // Z[k] = E + W_L^k O -> E's slot, Z[k + L/2] = E - W_L^k O -> O's slot
        const int za = G::zaddr(k);
        const cx<T> E = SE[za];
        const cx<T> WO = cmul(__ldg(p.tw + 2 * k), SO[za]);
        SE[za] = cadd(E, WO);
        SO[za] = csub(E, WO);
    }
    __syncthreads();
    auto Z = [&](int k) -> cx<T> { return k < LH ? SE[G::zaddr(k)] : SO[G::zaddr(k - LH)]; };
    const int NU = N / 2 + 1;
    const int i = (int)(row % N);
    const int pos = (i & 3) * (N >> 2) + (i >> 2);           // decimated by four for the column transform
    cx<T>* out = p.spec + (row / N) * (long long)NU * N + pos;
    const int kumax = __ldcg(p.ext);
    const int kend = kumax < L / 2 ? kumax : L / 2;
    for (int k = tid; k <= kend; k += G::NT) {               // untangle (factor 1/2 folded into the column pass)
        const cx<T> zk = Z(k), zm = Z((L - k) % L);
        const cx<T> E = mk<T>(zk.x + zm.x, zk.y - zm.y);
        const cx<T> O = mk<T>(zk.y + zm.y, zm.x - zk.x);
        const cx<T> WO = cmul(__ldg(p.tw + k), O);
        out[(long long)k * N] = cadd(E, WO);
        if (L - k <= kumax) { cx<T> xm = csub(E, WO); xm.y = -xm.y; out[(long long)(L - k) * N] = xm; }
    }
}

// The same row, split over a CLUSTER of two CTAs (nxy = 16384): CTA r of the pair transforms the samples 2 m + r
// of the packed sequence (one 4096-point transform, 256 threads, 70 KB: two CTAs of different rows fit an SM, so one
// row's load overlaps another row's arithmetic — the one-CTA form holds a whole SM and serialises them).  After a
// cluster barrier each CTA forms the outputs X[k] of its parity of k; the radix-2 combination and the untangle read
// E from the even CTA and O from the odd one, the partner's through distributed shared memory (`mapa` +
// `ld.shared::cluster`): four 16-byte reads per output, a few hundred outputs per row when the transform is pruned.
__device__ __forceinline__ uint32_t cluster_rank() { uint32_t r; asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r)); return r; }
__device__ __forceinline__ void cluster_barrier() {
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ uint32_t map_to_rank(uint32_t saddr, uint32_t rank) {
    uint32_t r; asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(saddr), "r"(rank)); return r;
}
__device__ __forceinline__ double2 ld_cluster(uint32_t addr, double) {
    double2 v; asm volatile("ld.shared::cluster.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(addr) : "memory"); return v;
}
__device__ __forceinline__ float2 ld_cluster(uint32_t addr, float) {
    float2 v; asm volatile("ld.shared::cluster.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(addr) : "memory"); return v;
}

template <typename T, int R1, int R2, int R3, bool SWEEP>
__global__ void __launch_bounds__(Geom<T, R1, R2, R3, 1>::NT, 2)
row_pass_c2_kernel(const RowParams<T> p) {
    using G = Geom<T, R1, R2, R3, 1>;
    constexpr int LH = G::L;                   // = N / 4: length of this CTA's transform
    constexpr int L = 2 * LH;                  // = N / 2: length of the packed complex row
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cx<T>* S = reinterpret_cast<cx<T>*>(smem_raw);
    const int t = threadIdx.x;
    const int N = p.N;
    const uint32_t r = cluster_rank();
    const long long row = blockIdx.x >> 1;
    if (!SWEEP && r == 0) prefetch_row_block(p, row, 1);
    pdl_wait();
    if (SWEEP) {
        const int i = (int)(row % N);
        fft_steps12<T, R1, R2, R3, G::TPF>(S, t, p.tw, 4, [&](int m) -> cx<T> {
            const int n = 2 * m + (int)r;
            return mk<T>((T)sweep_pixel<T>(p.sweep, N, i, 2 * n), (T)sweep_pixel<T>(p.sweep, N, i, 2 * n + 1));
        });
    } else {
        const cx<T>* z = reinterpret_cast<const cx<T>*>(p.image + row * (long long)N);
        fft_steps12<T, R1, R2, R3, G::TPF>(S, t, p.tw, 4, [&](int m) -> cx<T> { return __ldcs(z + 2 * m + (int)r); });
    }
    if (R3 > 1) {                              // step 3, in place
        for (int it = t; it < R1 * R2; it += G::TPF) {
            const int k1 = it % R1, c = it / R1;
            cx<T>* base = S + k1 * G::P1 + c * R3;
            cx<T> a[R3];
#pragma unroll
            for (int b = 0; b < R3; ++b) a[b] = base[b];
            Dft<T, R3>::run(a);
#pragma unroll
            for (int d = 0; d < R3; ++d) base[d] = a[d];
        }
    }
    cluster_barrier();                         // both halves complete and visible across the pair
    const uint32_t mine = smem_u32(S), theirs = map_to_rank(mine, r ^ 1u);
    const uint32_t sE = r == 0 ? mine : theirs, sO = r == 0 ? theirs : mine;
    // Z[k] = E[k] + W_L^k O[k] (k < L/2), Z[k + L/2] = E[k] - W_L^k O[k]
    auto Z = [&](int k) -> cx<T> {
        const int a = k < LH ? k : k - LH;
        const uint32_t off = (uint32_t)(G::zaddr(a) * sizeof(cx<T>));
        const cx<T> E = ld_cluster(sE + off, T()), O = ld_cluster(sO + off, T());
        const cx<T> WO = cmul(__ldg(p.tw + 2 * a), O);
        return k < LH ? cadd(E, WO) : csub(E, WO);
    };
    const int NU = N / 2 + 1;
    const int i = (int)(row % N);
    const int pos = (i & 3) * (N >> 2) + (i >> 2);           // decimated by four for the column transform
    cx<T>* out = p.spec + (row / N) * (long long)NU * N + pos;
    const int kumax = __ldcg(p.ext);
    const int kend = kumax < L / 2 ? kumax : L / 2;
    for (int k = 2 * t + (int)r; k <= kend; k += 2 * G::NT) {   // this CTA: k of its own parity; untangle as row_pass_x2
        const cx<T> zk = Z(k), zm = Z((L - k) % L);
        const cx<T> E = mk<T>(zk.x + zm.x, zk.y - zm.y);
        const cx<T> O = mk<T>(zk.y + zm.y, zm.x - zk.x);
        const cx<T> WO = cmul(__ldg(p.tw + k), O);
        out[(long long)k * N] = cadd(E, WO);
        if (L - k <= kumax) { cx<T> xm = csub(E, WO); xm.y = -xm.y; out[(long long)(L - k) * N] = xm; }
    }
    cluster_barrier();                         // the partner may still be reading this CTA's shared memory
}

// One quarter column (n1 = blockIdx.x & 3) per CTA: DFT_{N/4} in place, then times W_N^(n1 k2).
template <typename T, int R1, int R2, int R3>
__global__ void __launch_bounds__(Geom<T, R1, R2, R3, 1>::NT)
col_sub_kernel(const ColParams<T> p, cx<T>* __restrict__ work) {
    using G = Geom<T, R1, R2, R3, 1>;
    constexpr int LQ = G::L;                   // = N / 4
    constexpr int N = 4 * LQ, NU = N / 2 + 1;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cx<T>* S = reinterpret_cast<cx<T>*>(smem_raw);
    const int t = threadIdx.x;
    pdl_wait();
    const long long g = blockIdx.x >> 2;
    const int n1 = blockIdx.x & 3;
    if ((int)(g % NU) > __ldcg(p.ext)) return;
    cx<T>* q = work + g * (long long)N + (long long)n1 * LQ;
    fft_steps12<T, R1, R2, R3, G::TPF>(S, t, p.tw, 4, [&](int n) -> cx<T> { return q[n]; });
    for (int it = t; it < R1 * R2; it += G::TPF) {           // step 3 from shared memory, twiddle, straight to memory
        const int k1 = it % R1, c = it / R1;
        const cx<T>* base = S + k1 * G::P1 + c * R3;
        cx<T> a[R3];
#pragma unroll
        for (int b = 0; b < R3; ++b) a[b] = base[b];
        Dft<T, R3>::run(a);
#pragma unroll
        for (int d = 0; d < R3; ++d) {
            const int k2 = k1 + R1 * (c + R2 * d);
            q[k2] = n1 ? cmul(a[d], __ldg(p.tw + n1 * k2)) : a[d];
        }
    }
}

// X[k2 + (N/4) k1] = sum_n1 (-i)^(n1 k1) Y_n1[k2]  ->  spectrum (pairs or single copy), sign and row folds, pruned
template <typename T>
__global__ void __launch_bounds__(256) col_comb4_kernel(const ColParams<T> p) {
    const int N = p.N, LQ = N >> 2, NU = N / 2 + 1;
    pdl_wait();
    const int kumax = __ldcg(p.ext), rmin = __ldcg(p.ext + 1), rmax = __ldcg(p.ext + 2);
    const bool single = extent_is_whole_plane(p.ext, N);
    const long long g = blockIdx.y;
    const int ku = (int)(g % NU);
    if (ku > kumax) return;
    const cx<T>* col = p.work + g * (long long)N;
    NodePair<T>* own = p.pair + g * (long long)N;
    NodePair<T>* prev = own - (ku > 0 ? N : 0);
    cx<T>* sown = reinterpret_cast<cx<T>*>(p.pair) + g * (long long)N;
    for (int k2 = blockIdx.x * blockDim.x + threadIdx.x; k2 < LQ; k2 += gridDim.x * blockDim.x) {
        cx<T> a[4] = {col[k2], col[LQ + k2], col[2 * LQ + k2], col[3 * LQ + k2]};
        Dft<T, 4>::run(a);
        const T sgn = ((ku + k2) & 1) ? (T)-0.5 : (T)0.5;     // N/4 is even: kv and k2 have one parity
#pragma unroll
        for (int k1 = 0; k1 < 4; ++k1) {
            const int kvs = (k2 + k1 * LQ + N / 2) & (N - 1);
            if (kvs < rmin || kvs > rmax) continue;
            const cx<T> val = mk<T>(sgn * a[k1].x, sgn * a[k1].y);
            if (single) { sown[kvs] = val; } else { own[kvs].a = val; if (ku > 0) prev[kvs].b = val; }
        }
    }
}

// ------------------------------------------------------------------------------------------
// Standalone sweep (image written to memory) and the u-major -> paper-layout transpose.
// ------------------------------------------------------------------------------------------
template <typename T>
__global__ void sweep_kernel(SweepParams sp, int N, T* __restrict__ image) {
    const long long total = (long long)N * N;
    for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < total;
         idx += (long long)gridDim.x * blockDim.x) {
        const int i = (int)(idx / N), j = (int)(idx % N);
        image[idx] = (T)sweep_pixel<T>(sp, N, i, j);
    }
}

// out[kvs][ku] = single[ku][kvs]   (paper layout [N][N/2+1]; the whole-plane transform of
// gal_fft2_shifted_* leaves the spectrum in the single-copy layout)
template <typename T>
__global__ void transpose_to_paper_layout_kernel(const cx<T>* __restrict__ spec, cx<T>* __restrict__ out, int N) {
    __shared__ cx<T> tile[32][33];
    const int NU = N / 2 + 1;
    const int kv0 = blockIdx.x * 32, ku0 = blockIdx.y * 32;
    for (int r = threadIdx.y; r < 32; r += blockDim.y) {
        const int ku = ku0 + r, kv = kv0 + threadIdx.x;
        if (ku < NU && kv < N) tile[r][threadIdx.x] = spec[(long long)ku * N + kv];
    }
    __syncthreads();
    for (int r = threadIdx.y; r < 32; r += blockDim.y) {
        const int kv = kv0 + r, ku = ku0 + threadIdx.x;
        if (ku < NU && kv < N) out[(long long)kv * NU + ku] = tile[threadIdx.x][r];
    }
}

}  // namespace galb
