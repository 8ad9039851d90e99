// galario_oracle.cpp — CPU ORACLE for the GALARIO hot path (arXiv:1709.06999).
//
// THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
// and the cpu_baseline / --impl reference legs of bench.py may load it.  It shares no
// code, header, table or helper with the CUDA path in paper_1709_06999_b200/csrc/.
//
// It is deliberately plain and slow: it follows the paper's own numpy/scipy listing
// (Appendix D) step by step, in the listing's order and notation,
// with a naive radix-2 FFT (direct DFT for nxy <= 64) standing in for numpy's rfft2.
// No blocking, no fusion, no reordering.  Every function cites the passage it follows.
//
// Readings of the paper where it is silent or garbled are the ones listed in
// DESIGN.md ("Readings", items A1..A20; they restate SURVEY.md §8(c)).
//
// Pins (tests/test_oracle_*.py, run with -m "not gpu"): brute-force sky-coordinate DFT
// at nxy <= 64, the Appendix-D listing re-run with numpy.fft + scipy, delta-source and
// Gaussian closed forms, Hermitian symmetry, Parseval, PA = 90 deg identity, chi2
// invariants, scipy.interp1d for the sweep; the Hankel evaluation (H1) by the Gaussian and uniform-disc
// closed forms, an elliptical Gaussian (inclination, PA), scipy quadrature and the paper's own 1e-5
// agreement with sampleProfile.  No function here is "parity unpinned".
//
// Build: g++ -O2 -ffp-contract=off -std=c++17 -shared -fPIC -pthread galario_oracle.cpp -o liboracle.so
//
// All pointers are HOST pointers, all arrays are double, caller-owned.  Complex arrays
// are interleaved (re, im).  Functions return 0 on success, negative on bad arguments.

#include <cmath>
#include <complex>
#include <cstdint>
#include <cstring>
#include <thread>
#include <vector>
#include <algorithm>

namespace {

template <typename T> struct Pi;
template <> struct Pi<double>      { static double v()      { return 3.14159265358979323846; } };
template <> struct Pi<long double> { static long double v() { return 3.14159265358979323846264338327950288L; } };

inline bool is_pow2(int n) { return n > 0 && (n & (n - 1)) == 0; }

// Floor modulo: result in [0, n).
inline int64_t fmod_i(int64_t a, int64_t n) { int64_t r = a % n; return r < 0 ? r + n : r; }

// Run f(t, begin, end) over [0, n) split in `nthreads` contiguous chunks (thread order fixed).
template <typename F>
void parallel_chunks(int64_t n, int nthreads, F f) {
    if (nthreads <= 1 || n < 2) { f(0, (int64_t)0, n); return; }
    int T = (int)std::min<int64_t>(nthreads, n);
    std::vector<std::thread> th;
    for (int t = 0; t < T; ++t) {
        int64_t b = n * t / T, e = n * (t + 1) / T;
        th.emplace_back([=] { f(t, b, e); });
    }
    for (auto& x : th) x.join();
}

// ---------------------------------------------------------------------------------------
// O3 (1-D building block).  Discrete Fourier transform with the kernel of numpy's forward
// FFT, exp(-2 pi i k n / N) (np.fft.rfft2).
// ---------------------------------------------------------------------------------------

// Twiddle table w[m] = exp(-2 pi i m / N), m = 0..N-1, each entry evaluated directly.
template <typename T>
std::vector<std::complex<T>> twiddles(int N) {
    std::vector<std::complex<T>> w(N);
    for (int m = 0; m < N; ++m) {
        T a = -2 * Pi<T>::v() * (T)m / (T)N;
        w[m] = std::complex<T>(std::cos(a), std::sin(a));
    }
    return w;
}

// Textbook iterative radix-2 decimation-in-time FFT, in place, stride 1 (Cooley & Tukey 1965,
// the algorithm PAPER.md:236 names).  N must be a power of two.
template <typename T>
void fft_radix2(std::complex<T>* x, int N, const std::vector<std::complex<T>>& w) {
    // bit reversal permutation
    for (int i = 1, j = 0; i < N; ++i) {
        int bit = N >> 1;
        for (; j & bit; bit >>= 1) j ^= bit;
        j ^= bit;
        if (i < j) std::swap(x[i], x[j]);
    }
    for (int len = 2; len <= N; len <<= 1) {
        int half = len >> 1, step = N / len;
        for (int s = 0; s < N; s += len)
            for (int k = 0; k < half; ++k) {
                std::complex<T> t = x[s + k + half] * w[k * step];
                std::complex<T> a = x[s + k];
                x[s + k] = a + t;
                x[s + k + half] = a - t;
            }
    }
}

// ---------------------------------------------------------------------------------------
// O2 + O3 + O4:  fft_r2c_shifted = fftshift( rfft2( fftshift(image) ), axes=0 )
// (PAPER.md:659).  Output G[N][N/2+1], row index = v (zero frequency at row N/2),
// column index = u >= 0.
// ---------------------------------------------------------------------------------------
template <typename T>
int spectrum_T(const double* image, int N, std::complex<T>* G, int nthreads) {
    if (!image || !G || N < 2 || (N & 1)) return -1;
    const int H = N / 2, NU = N / 2 + 1;

    // O2: S = fftshift(image) on both axes: S[i'][j'] = A[(i'+N/2)%N][(j'+N/2)%N].
    std::vector<T> S((size_t)N * N);
    for (int i = 0; i < N; ++i)
        for (int j = 0; j < N; ++j)
            S[(size_t)i * N + j] = (T)image[(size_t)((i + H) % N) * N + (j + H) % N];

    std::vector<std::complex<T>> F((size_t)N * NU);  // F[kv][ku], unshifted rfft2 output

    if (N <= 64 || !is_pow2(N)) {
        // O3, tiny images: the 2-D DFT definition written out,
        // F[kv][ku] = sum_{i',j'} S[i'][j'] exp(-2 pi i (kv i' + ku j') / N).
        auto w = twiddles<T>(N);
        for (int kv = 0; kv < N; ++kv)
            for (int ku = 0; ku < NU; ++ku) {
                std::complex<T> acc(0, 0);
                for (int i = 0; i < N; ++i)
                    for (int j = 0; j < N; ++j)
                        acc += S[(size_t)i * N + j] * w[(int)(((int64_t)kv * i + (int64_t)ku * j) % N)];
                F[(size_t)kv * NU + ku] = acc;
            }
    } else {
        // O3, N >= 128: naive radix-2 FFT of every row (real data promoted to complex, the
        // ku <= N/2 half kept), then of every column.  No real-input shortcut is taken.
        auto w = twiddles<T>(N);
        parallel_chunks(N, nthreads, [&](int, int64_t b, int64_t e) {
            std::vector<std::complex<T>> row(N);
            for (int64_t i = b; i < e; ++i) {
                for (int j = 0; j < N; ++j) row[j] = std::complex<T>(S[(size_t)i * N + j], 0);
                fft_radix2(row.data(), N, w);
                for (int ku = 0; ku < NU; ++ku) F[(size_t)i * NU + ku] = row[ku];
            }
        });
        parallel_chunks(NU, nthreads, [&](int, int64_t b, int64_t e) {
            std::vector<std::complex<T>> col(N);
            for (int64_t ku = b; ku < e; ++ku) {
                for (int i = 0; i < N; ++i) col[i] = F[(size_t)i * NU + ku];
                fft_radix2(col.data(), N, w);
                for (int kv = 0; kv < N; ++kv) F[(size_t)kv * NU + ku] = col[kv];
            }
        });
    }

    // O4: fftshift along axis 0 only: G[(kv+N/2)%N][ku] = F[kv][ku].
    for (int kv = 0; kv < N; ++kv)
        std::memcpy((void*)&G[(size_t)((kv + H) % N) * NU], (const void*)&F[(size_t)kv * NU],
                    sizeof(std::complex<T>) * NU);
    return 0;
}

// Node of the shifted half-plane spectrum, extended to ALL integer (row, col) by the
// periodicity and Hermitian symmetry of the DFT of a real image (reading A6).
// Inside 0 <= row < N, 0 <= col <= N/2 this is G[row][col] itself, so nothing changes for
// points Appendix D can address.
template <typename T>
inline std::complex<T> node(const std::complex<T>* G, int N, int64_t row, int64_t col) {
    const int H = N / 2, NU = N / 2 + 1;
    int64_t kv = row - H;              // signed v frequency index of this row
    int64_t cu = fmod_i(col, N);       // u frequency index folded to [0, N)
    if (cu <= H) {
        int64_t r = fmod_i(fmod_i(kv, N) + H, N);
        return G[(size_t)r * NU + cu];
    }
    // F[kv][ku] = conj F[-kv][-ku] for a real image.
    int64_t r = fmod_i(fmod_i(-kv, N) + H, N);
    return std::conj(G[(size_t)r * NU + (N - cu)]);
}

// ---------------------------------------------------------------------------------------
// O5 + O6 + O7: rotate the uv points, interpolate the spectrum bilinearly, apply the phase
// (Eq. 11-13).
// ---------------------------------------------------------------------------------------
template <typename T>
int sample_spectrum_T(const std::complex<T>* G, int N, double dxy_, const double* u, const double* v,
                      int64_t M, double dRA_, double dDec_, double PA_, double* vis, int64_t* oob_out,
                      int nthreads) {
    if (!G || N < 2 || (N & 1) || M < 0 || !(dxy_ > 0)) return -1;
    if (M > 0 && (!u || !v || !vis)) return -1;
    const T dxy = (T)dxy_;
    // PAPER.md:653-655:  dRA *= 2 pi ; dDec *= 2 pi ; du = 1 / (nxy * dxy)
    const T dRA = (T)dRA_ * 2 * Pi<T>::v();
    const T dDec = (T)dDec_ * 2 * Pi<T>::v();
    const T du = 1 / ((T)N * dxy);
    // PAPER.md:662-663.  cos/sin of PA are taken once, in double (reading A16), so that both
    // sides of a parity test use the same two numbers.
    const T cos_PA = (T)std::cos(PA_);
    const T sin_PA = (T)std::sin(PA_);
    // PAPER.md:669-670
    const T dRArot = dRA * cos_PA - dDec * sin_PA;
    const T dDecrot = dRA * sin_PA + dDec * cos_PA;

    std::vector<int64_t> oob_part(std::max(1, nthreads), 0);
    parallel_chunks(M, nthreads, [&](int t, int64_t b, int64_t e) {
        int64_t oob = 0;
        for (int64_t k = b; k < e; ++k) {
            // PAPER.md:667-668 (Eq. 11-12)
            const T urot = (T)u[k] * cos_PA - (T)v[k] * sin_PA;
            const T vrot = (T)u[k] * sin_PA + (T)v[k] * cos_PA;
            // interpolation indices; Hermitian fold for urot < 0.
            const T urot_idx = std::fabs(urot) / du;
            const bool uneg = urot < 0;
            const T vrot_idx = uneg ? (T)N / 2 - vrot / du : (T)N / 2 + vrot / du;
            if (urot_idx > (T)(N / 2) || vrot_idx < 0 || vrot_idx > (T)(N - 1)) ++oob;
            // RectBivariateSpline(kx=ky=1).ev == bilinear interpolation on the
            // grid rows 0..N-1, columns 0..N/2, Re and Im separately.
            const T fx0 = std::floor(urot_idx), fy0 = std::floor(vrot_idx);
            const int64_t ix = (int64_t)fx0, iy = (int64_t)fy0;
            const T tx = urot_idx - fx0, ty = vrot_idx - fy0;
            const std::complex<T> g00 = node(G, N, iy, ix), g01 = node(G, N, iy, ix + 1);
            const std::complex<T> g10 = node(G, N, iy + 1, ix), g11 = node(G, N, iy + 1, ix + 1);
            T ReInt = (1 - ty) * ((1 - tx) * g00.real() + tx * g01.real()) +
                      ty * ((1 - tx) * g10.real() + tx * g11.real());
            T ImInt = (1 - ty) * ((1 - tx) * g00.imag() + tx * g01.imag()) +
                      ty * ((1 - tx) * g10.imag() + tx * g11.imag());
            // ImInt[uneg] *= -1.
            if (uneg) ImInt = -ImInt;
            // theta = urot*dRArot + vrot*dDecrot ; vis = (Re + i Im)(cos + i sin)
            const T theta = urot * dRArot + vrot * dDecrot;
            const T c = std::cos(theta), s = std::sin(theta);
            vis[2 * k] = (double)(ReInt * c - ImInt * s);
            vis[2 * k + 1] = (double)(ReInt * s + ImInt * c);
        }
        oob_part[t] = oob;
    });
    if (oob_out) { int64_t s = 0; for (auto x : oob_part) s += x; *oob_out = s; }
    return 0;
}

// ---------------------------------------------------------------------------------------
// O8: chi2 = sum(((vis.real - vis_obs_re)**2 + (vis.imag - vis_obs_im)**2) * weights)
// (Eq. 10 at PAPER.md:196).  Accumulated in long double, in index order
// (per-thread partials added in thread order when nthreads > 1).
// ---------------------------------------------------------------------------------------
double chi2_of(const double* vis, const double* re_obs, const double* im_obs, const double* w, int64_t M,
               int nthreads) {
    std::vector<long double> part(std::max(1, nthreads), 0.0L);
    parallel_chunks(M, nthreads, [&](int t, int64_t b, int64_t e) {
        long double acc = 0;
        for (int64_t k = b; k < e; ++k) {
            long double dr = (long double)vis[2 * k] - re_obs[k];
            long double di = (long double)vis[2 * k + 1] - im_obs[k];
            acc += (dr * dr + di * di) * (long double)w[k];
        }
        part[t] = acc;
    });
    long double s = 0;
    for (auto x : part) s += x;
    return (double)s;
}

// ---------------------------------------------------------------------------------------
// O1: sweep.  x, y meshes run from +0.5 to -0.5 + 1/N times N*dxy
// (PAPER.md:738-739), radius sqrt((x/cos inc)^2 + y^2), profile * dxy^2
// (PAPER.md:745), linear interpolation on gridrad with fill_value = 0 outside
// [Rmin, Rmin + dR (nr-1)].  No special central pixel (reading A5).
// ---------------------------------------------------------------------------------------
template <typename T>
int sweep_T(const double* I, int nr, double Rmin_, double dR_, int N, double dxy_, double inc_, double* image) {
    if (!I || !image || nr < 2 || N < 1 || !(dR_ > 0) || !(dxy_ > 0)) return -1;
    const T Rmin = (T)Rmin_, dR = (T)dR_, dxy = (T)dxy_;
    const T inc_cos = (T)std::cos(inc_);
    if (!(inc_cos > 0)) return -1;
    const T Rmax = Rmin + dR * (T)(nr - 1);
    for (int i = 0; i < N; ++i) {
        // np.linspace(0.5, -0.5 + 1/N, N)[i] = 0.5 - i/N  (step -1/N)
        const T y = ((T)0.5 - (T)i / (T)N) * dxy * (T)N;
        for (int j = 0; j < N; ++j) {
            const T x = ((T)0.5 - (T)j / (T)N) * dxy * (T)N;
            const T xs = x / inc_cos;
            const T r = std::sqrt(xs * xs + y * y);
            T val = 0;
            if (r >= Rmin && r <= Rmax) {
                T pos = (r - Rmin) / dR;
                int64_t k = (int64_t)std::floor(pos);
                if (k >= nr - 1) k = nr - 2;  // r == Rmax: last interval, weight 1 on the last sample
                if (k < 0) k = 0;
                const T t = pos - (T)k;
                val = ((T)I[k] + t * ((T)I[k + 1] - (T)I[k])) * dxy * dxy;
            }
            image[(size_t)i * N + j] = (double)val;
        }
    }
    return 0;
}

// ---------------------------------------------------------------------------------------
// H1: direct Hankel-transform evaluation of an axisymmetric profile (Eq. 25)
//       V(rho) = 2 pi int_0^inf I(r) J0(2 pi rho r) r dr,   rho = deprojected uv distance,
// the analytic result the paper checks sampleProfile against, offered as an
// alternative to sweep + FFT + interpolation for axisymmetric models.
// Readings (A20): the profile is the one the sweep uses — samples I[k] at
// R_k = Rmin + k dR, zero outside [Rmin, Rmax]; the integral is the
// composite trapezoid rule on that grid; the sweep stretches the East-West axis by 1/cos inc
// (PAPER.md:740), so by the scaling theorem the transform is cos(inc) V(rho) at
// rho = sqrt((u' cos inc)^2 + v'^2); (u', v') and the phase follow the listing
// exactly as in sample_spectrum_T.  J0 is the standard library's
// std::cyl_bessel_j(0, x).  The result is real before the phase factor.
// ---------------------------------------------------------------------------------------
int hankel_sample(const double* I, int nr, double Rmin, double dR, const double* u, const double* v, int64_t M,
                  double dRA, double dDec, double PA, double inc, double* vis, int nthreads) {
    if (!I || nr < 2 || !(dR > 0) || M < 0 || (M > 0 && (!u || !v || !vis))) return -1;
    const double inc_cos = std::cos(inc);
    if (!(inc_cos > 0)) return -1;
    const double pi = Pi<double>::v();
    const double cos_PA = std::cos(PA), sin_PA = std::sin(PA);
    dRA *= 2 * pi;
    dDec *= 2 * pi;
    const double dRArot = dRA * cos_PA - dDec * sin_PA;
    const double dDecrot = dRA * sin_PA + dDec * cos_PA;
    parallel_chunks(M, nthreads, [&](int, int64_t b, int64_t e) {
        for (int64_t k = b; k < e; ++k) {
            const double urot = u[k] * cos_PA - v[k] * sin_PA;
            const double vrot = u[k] * sin_PA + v[k] * cos_PA;
            const double rho = std::sqrt((urot * inc_cos) * (urot * inc_cos) + vrot * vrot);
            long double acc = 0;
            for (int j = 0; j < nr; ++j) {
                const double r = Rmin + dR * (double)j;
                const double term = I[j] * std::cyl_bessel_j(0.0, 2 * pi * rho * r) * r;
                acc += (j == 0 || j == nr - 1) ? 0.5L * term : (long double)term;
            }
            const double V = 2 * pi * inc_cos * dR * (double)acc;
            const double theta = urot * dRArot + vrot * dDecrot;
            vis[2 * k] = V * std::cos(theta);
            vis[2 * k + 1] = V * std::sin(theta);
        }
    });
    return 0;
}

}  // namespace

// =========================================================================================
// C ABI
// =========================================================================================
extern "C" {

// O1.  image[nxy][nxy] <- sweep of profile I[nr] (Jy/sr) on R_k = Rmin + k dR.
int orc_sweep(const double* I, int nr, double Rmin, double dR, int nxy, double dxy, double inc, double* image) {
    return sweep_T<double>(I, nr, Rmin, dR, nxy, dxy, inc, image);
}

// O2+O3+O4.  G[nxy][nxy/2+1] complex interleaved <- fftshift(rfft2(fftshift(image)), axes=0).
int orc_spectrum(const double* image, int nxy, double* G, int nthreads) {
    return spectrum_T<double>(image, nxy, reinterpret_cast<std::complex<double>*>(G), nthreads);
}

// Same, carried in long double and rounded to double on output (self-validation of O3).
int orc_spectrum_ld(const double* image, int nxy, double* G, int nthreads) {
    if (nxy < 2) return -1;
    std::vector<std::complex<long double>> Gl((size_t)nxy * (nxy / 2 + 1));
    int rc = spectrum_T<long double>(image, nxy, Gl.data(), nthreads);
    if (rc) return rc;
    for (size_t k = 0; k < Gl.size(); ++k) { G[2 * k] = (double)Gl[k].real(); G[2 * k + 1] = (double)Gl[k].imag(); }
    return 0;
}

// O5+O6+O7 on a spectrum produced by orc_spectrum.  vis[2M] interleaved.  oob (may be null)
// receives the number of points whose interpolation cell leaves the half-plane grid.
int orc_sample_spectrum(const double* G, int nxy, double dxy, const double* u, const double* v, int64_t M,
                        double dRA, double dDec, double PA, double* vis, int64_t* oob, int nthreads) {
    return sample_spectrum_T<double>(reinterpret_cast<const std::complex<double>*>(G), nxy, dxy, u, v, M, dRA,
                                     dDec, PA, vis, oob, nthreads);
}

// O8.
double orc_chi2(const double* vis, const double* re_obs, const double* im_obs, const double* w, int64_t M,
                int nthreads) {
    return chi2_of(vis, re_obs, im_obs, w, M, nthreads);
}

// sampleImage = O2..O7.
int orc_sample_image(const double* image, int nxy, double dxy, const double* u, const double* v, int64_t M,
                     double dRA, double dDec, double PA, double* vis, int64_t* oob, int nthreads) {
    if (nxy < 2 || (nxy & 1)) return -1;
    std::vector<std::complex<double>> G((size_t)nxy * (nxy / 2 + 1));
    int rc = spectrum_T<double>(image, nxy, G.data(), nthreads);
    if (rc) return rc;
    return sample_spectrum_T<double>(G.data(), nxy, dxy, u, v, M, dRA, dDec, PA, vis, oob, nthreads);
}

// The whole sampleImage carried in long double (inputs/outputs double).
int orc_sample_image_ld(const double* image, int nxy, double dxy, const double* u, const double* v, int64_t M,
                        double dRA, double dDec, double PA, double* vis, int64_t* oob, int nthreads) {
    if (nxy < 2 || (nxy & 1)) return -1;
    std::vector<std::complex<long double>> G((size_t)nxy * (nxy / 2 + 1));
    int rc = spectrum_T<long double>(image, nxy, G.data(), nthreads);
    if (rc) return rc;
    return sample_spectrum_T<long double>(G.data(), nxy, dxy, u, v, M, dRA, dDec, PA, vis, oob, nthreads);
}

// chi2Image = O2..O8.
int orc_chi2_image(const double* image, int nxy, double dxy, const double* u, const double* v,
                   const double* re_obs, const double* im_obs, const double* w, int64_t M, double dRA,
                   double dDec, double PA, double* chi2, int64_t* oob, int nthreads) {
    if (!chi2 || M < 0) return -1;
    std::vector<double> vis((size_t)2 * std::max<int64_t>(M, 1));
    int rc = orc_sample_image(image, nxy, dxy, u, v, M, dRA, dDec, PA, vis.data(), oob, nthreads);
    if (rc) return rc;
    *chi2 = chi2_of(vis.data(), re_obs, im_obs, w, M, nthreads);
    return 0;
}

// sampleProfile = O1 then sampleImage.
int orc_sample_profile(const double* I, int nr, double Rmin, double dR, int nxy, double dxy, const double* u,
                       const double* v, int64_t M, double dRA, double dDec, double PA, double inc, double* vis,
                       int64_t* oob, int nthreads) {
    if (nxy < 2) return -1;
    std::vector<double> image((size_t)nxy * nxy);
    int rc = sweep_T<double>(I, nr, Rmin, dR, nxy, dxy, inc, image.data());
    if (rc) return rc;
    return orc_sample_image(image.data(), nxy, dxy, u, v, M, dRA, dDec, PA, vis, oob, nthreads);
}

// chi2Profile = O1 then chi2Image.
int orc_chi2_profile(const double* I, int nr, double Rmin, double dR, int nxy, double dxy, const double* u,
                     const double* v, const double* re_obs, const double* im_obs, const double* w, int64_t M,
                     double dRA, double dDec, double PA, double inc, double* chi2, int64_t* oob, int nthreads) {
    if (nxy < 2) return -1;
    std::vector<double> image((size_t)nxy * nxy);
    int rc = sweep_T<double>(I, nr, Rmin, dR, nxy, dxy, inc, image.data());
    if (rc) return rc;
    return orc_chi2_image(image.data(), nxy, dxy, u, v, re_obs, im_obs, w, M, dRA, dDec, PA, chi2, oob, nthreads);
}

// Batched cube (reading A17; not in the paper): C independent chi2Image problems sharing
// (nxy, dxy, dRA, dDec, PA, M); arrays are [C][...] contiguous; chi2_total = sum in channel order.
int orc_chi2_image_batch(const double* images, int C, int nxy, double dxy, const double* u, const double* v,
                         const double* re_obs, const double* im_obs, const double* w, int64_t M, double dRA,
                         double dDec, double PA, double* chi2_per_channel, double* chi2_total, int64_t* oob,
                         int nthreads) {
    if (C < 0 || !chi2_per_channel) return -1;
    long double tot = 0;
    int64_t oob_all = 0;
    for (int c = 0; c < C; ++c) {
        int64_t o = 0;
        int rc = orc_chi2_image(images + (size_t)c * nxy * nxy, nxy, dxy, u + (size_t)c * M, v + (size_t)c * M,
                                re_obs + (size_t)c * M, im_obs + (size_t)c * M, w + (size_t)c * M, M, dRA, dDec,
                                PA, &chi2_per_channel[c], &o, nthreads);
        if (rc) return rc;
        tot += chi2_per_channel[c];
        oob_all += o;
    }
    if (chi2_total) *chi2_total = (double)tot;
    if (oob) *oob = oob_all;
    return 0;
}

// H1.  sampleProfile by the direct Hankel transform of Eq. 25; vis[2M] interleaved.
int orc_sample_profile_hankel(const double* I, int nr, double Rmin, double dR, const double* u, const double* v,
                              int64_t M, double dRA, double dDec, double PA, double inc, double* vis, int nthreads) {
    return hankel_sample(I, nr, Rmin, dR, u, v, M, dRA, dDec, PA, inc, vis, nthreads);
}

// chi2Profile by the same evaluation = H1 then O8.
int orc_chi2_profile_hankel(const double* I, int nr, double Rmin, double dR, const double* u, const double* v,
                            const double* re_obs, const double* im_obs, const double* w, int64_t M, double dRA,
                            double dDec, double PA, double inc, double* chi2, int nthreads) {
    if (!chi2 || M < 0) return -1;
    std::vector<double> vis((size_t)2 * std::max<int64_t>(M, 1));
    int rc = hankel_sample(I, nr, Rmin, dR, u, v, M, dRA, dDec, PA, inc, vis.data(), nthreads);
    if (rc) return rc;
    *chi2 = chi2_of(vis.data(), re_obs, im_obs, w, M, nthreads);
    return 0;
}

}  // extern "C"
