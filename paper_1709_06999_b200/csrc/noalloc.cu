// noalloc.cu — gal_chi2_profile_hankel_noalloc_f64: chi2Profile by the direct Hankel transform (Eq. 25,
// PAPER.md:366-368; chi2 of Eq. 10) for callers that must not allocate device memory.
//
// Who this is for.  Every other entry point needs a gal_plan, and gal_plan_create calls cudaMalloc several times
// (workspace, tables, reduction scratch).  Some users of this library cannot afford that:
//   * a fitting code that was handed a fixed slice of the GPU by its host application (an arena carved out once at
//     start-up, a memory-capped MPS client, a GPU whose 180 GB are already spoken for by the walkers of a large
//     run): a cudaMalloc there fails, or takes memory somebody else was promised;
//   * a latency-critical loop: cudaMalloc and cudaFree synchronise the whole device and take the driver's
//     allocator lock, which stalls every other stream of the process.
// For them this file offers one call with no plan behind it.  It calls no cudaMalloc, cudaFree, cudaMallocAsync
// or any other allocating routine, now or at set-up; the caller passes inputs and the output as device pointers.
//
// Where the scratch lives.  The deterministic chi2 reduction needs one double per CTA and a ticket counter.  They
// sit in the file-scope array `noalloc_scratch` below: 64 KiB + 256 B of device memory that EVERY GPU which loads
// this library holds from module load until the process exits, used or not.  Its fixed size is what limits the
// call: one CTA sums NOALLOC_TILE = 128 points, the array has room for GAL_NOALLOC_MAX_POINTS / 128 = 8192
// partial sums, so M above GAL_NOALLOC_MAX_POINTS = 1 048 576 is refused with GAL_ERR_TOO_LARGE (nothing is
// launched).  Longer sets go through gal_chi2_profile_hankel_f64 on a plan, or are split by the caller (chi2 is
// additive over points).
//
// Set-up.  In host code the name `noalloc_scratch` is only a handle of the runtime, not a device address (a
// kernel handed `noalloc_scratch` from the host would fault or scribble over unrelated memory).  The first call
// on each device therefore asks the runtime for the real address — cudaGetSymbolAddress with that device current,
// return code checked — and caches it per device; later calls reuse it.  That first call loads this module's
// kernels and data onto the device as a side effect: make it once, ahead of time, before any stream capture is
// begun and before the latency-critical part of the program.
//
// Sharing.  There is one array per device and every call on that device uses it.  The ticket counter is set to
// zero on the caller's stream in front of every launch (so a call that was aborted half-way cannot poison the
// next one); the partial sums need no clearing, each launch writes every slot it later reads.  The array keeps
// the last call's partial sums afterwards.  Two calls whose kernels may overlap on the same GPU — different
// streams, different host threads — race on it and return garbage: issue the calls to one stream, or order
// them yourself with events.  (Calls on different GPUs do not interact.)
//
// The arithmetic per point is that of hankel.cuh's kernel (rotation, trapezoid rule over the profile with the
// hand-written J0, cos(inc) factor, phase ramp in turns, chi2 term), only the summation order differs: fixed
// tiles of 128 points per CTA whatever the GPU, partial sums added in tile order by the last CTA to finish.  The
// result is therefore bit-reproducible from run to run AND from one GPU model to another.
#include "../../include/galario_b200.h"

#include <cmath>
#include <mutex>

#include "hankel.cuh"

namespace {

using namespace galb;

constexpr int NOALLOC_WARPS = 8;                 // per CTA
constexpr int NOALLOC_PER_WARP = 16;             // points per warp
constexpr int NOALLOC_TILE = NOALLOC_WARPS * NOALLOC_PER_WARP;                     // 128 points per CTA
constexpr long long NOALLOC_MAX_TILES = GAL_NOALLOC_MAX_POINTS / NOALLOC_TILE;     // 8192 partial sums
constexpr size_t NOALLOC_CTRL_BYTES = 256;       // [0] u32 ticket; the rest is padding up to the alignment
constexpr size_t NOALLOC_SCRATCH_BYTES = NOALLOC_CTRL_BYTES + sizeof(double) * NOALLOC_MAX_TILES;
static_assert(GAL_NOALLOC_MAX_POINTS % NOALLOC_TILE == 0, "whole tiles");
static_assert(NOALLOC_SCRATCH_BYTES == 65792, "the size the header and the README state");

// The scratch of every call on this device: [ticket | pad to 256 B | double partial[8192]].
static __device__ __align__(256) unsigned char noalloc_scratch[NOALLOC_SCRATCH_BYTES];

// `scratch` is the DEVICE address of noalloc_scratch (cudaGetSymbolAddress, below).
__global__ void __launch_bounds__(NOALLOC_WARPS * 32)
hankel_chi2_noalloc_kernel(const HankelParams h, const double* __restrict__ u, const double* __restrict__ v,
                           const double* __restrict__ re_obs, const double* __restrict__ im_obs,
                           const double* __restrict__ w, const long long M, unsigned char* scratch,
                           double* __restrict__ chi2_out) {
    unsigned int* ticket = reinterpret_cast<unsigned int*>(scratch);
    double* partial = reinterpret_cast<double*>(scratch + NOALLOC_CTRL_BYTES);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const double* __restrict__ I = (const double*)h.I;
    __shared__ double wsum[NOALLOC_WARPS];
    __shared__ bool is_last;

    double acc = 0.0;
    const long long k0 = (long long)blockIdx.x * NOALLOC_TILE + wid * NOALLOC_PER_WARP;
    for (int i = 0; i < NOALLOC_PER_WARP; ++i) {
        const long long k = k0 + i;
        if (k >= M) break;                                   // (uniform over the warp)
        const double uk = __ldg(u + k), vk = __ldg(v + k);
        const double urot = __dsub_rn(__dmul_rn(uk, h.cos_PA), __dmul_rn(vk, h.sin_PA));
        const double vrot = __dadd_rn(__dmul_rn(uk, h.sin_PA), __dmul_rn(vk, h.cos_PA));
        const double ud = urot * h.inc_cos;                  // the sweep stretches East-West
        const double rho = sqrt(fma(ud, ud, vrot * vrot));
        double s = 0.0;                                      // trapezoid rule on R_j = Rmin + j dR
        for (int j = lane; j < h.nr; j += 32) {
            const double r = fma(h.dR, (double)j, h.Rmin);
            double term = __ldg(I + j) * bessel_j0_turns(rho * r) * r;
            if (j == 0 || j == h.nr - 1) term *= 0.5;
            s += term;
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
        const double V = 6.283185307179586477 * h.inc_cos * h.dR * s;
        double vr = V, vi = 0.0;
        if (h.has_phase) {
            int q;
            const double a = quarter_reduce(fma(urot, h.dRA_turns, vrot * h.dDec_turns), &q);
            double sn, cs;
            sincos_quarter(a, q, &sn, &cs);
            vr = V * cs;
            vi = V * sn;
        }
        if (lane == 0) {                                     // PAPER.md:718 (Eq. 10)
            const double dr = vr - __ldg(re_obs + k), di = vi - __ldg(im_obs + k);
            acc += fma(dr, dr, di * di) * __ldg(w + k);
        }
    }
    // CTA sum in warp order -> this tile's slot -> the last CTA to take a ticket adds the slots in tile order
    if (lane == 0) wsum[wid] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = 0.0;
        for (int i = 0; i < NOALLOC_WARPS; ++i) s += wsum[i];
        partial[blockIdx.x] = s;
        __threadfence();
        is_last = (atomicAdd(ticket, 1u) == gridDim.x - 1);
    }
    __syncthreads();
    if (!is_last) return;
    __threadfence();
    const volatile double* part = partial;
    double s = 0.0;
    for (int i = threadIdx.x; i < (int)gridDim.x; i += blockDim.x) s += part[i];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_down_sync(0xffffffffu, s, o);
    if (lane == 0) wsum[wid] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        double tot = 0.0;
        for (int i = 0; i < NOALLOC_WARPS; ++i) tot += wsum[i];
        *chi2_out = tot;
        *ticket = 0u;                                        // (the next call clears it again on its stream)
    }
}

// Device address of noalloc_scratch, looked up once per device.
constexpr int NOALLOC_MAX_DEVICES = 64;
std::mutex noalloc_mu;
unsigned char* noalloc_addr[NOALLOC_MAX_DEVICES] = {};
int noalloc_last_cuda = 0;

// Call with `device` current.  No allocation: the array exists since the module was loaded on this device.
int noalloc_scratch_address(int device, unsigned char** out) {
    std::lock_guard<std::mutex> lock(noalloc_mu);
    if (!noalloc_addr[device]) {
        void* ptr = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&ptr, noalloc_scratch);
        if (e != cudaSuccess || !ptr) {
            noalloc_last_cuda = (int)e;
            return GAL_ERR_CUDA;
        }
        noalloc_addr[device] = static_cast<unsigned char*>(ptr);
    }
    *out = noalloc_addr[device];
    return GAL_OK;
}

int noalloc_fail(cudaError_t e) {
    std::lock_guard<std::mutex> lock(noalloc_mu);
    noalloc_last_cuda = (int)e;
    return GAL_ERR_CUDA;
}

}  // namespace

extern "C" {

int gal_noalloc_last_cuda_error(void) {
    std::lock_guard<std::mutex> lock(noalloc_mu);
    return noalloc_last_cuda;
}

size_t gal_noalloc_scratch_bytes(void) { return NOALLOC_SCRATCH_BYTES; }

int gal_chi2_profile_hankel_noalloc_f64(int device, const double* I, int nr, double Rmin, double dR, const double* u,
                                        const double* v, const double* re_obs, const double* im_obs, const double* w,
                                        int64_t M, double dRA, double dDec, double PA, double inc, double* chi2_out,
                                        void* stream) {
    if (device < 0 || device >= NOALLOC_MAX_DEVICES || !I || nr < 2 || !(dR > 0) || !std::isfinite(Rmin) || !chi2_out || M < 0)
        return GAL_ERR_INVALID_ARGUMENT;
    if (!std::isfinite(inc) || !(std::fabs(inc) < 1.5707963267948966) || !(std::cos(inc) > 0)) return GAL_ERR_INVALID_ARGUMENT;
    if (!std::isfinite(dRA) || !std::isfinite(dDec) || !std::isfinite(PA)) return GAL_ERR_INVALID_ARGUMENT;
    if (M > 0 && (!u || !v || !re_obs || !im_obs || !w)) return GAL_ERR_INVALID_ARGUMENT;
    if (M > (int64_t)GAL_NOALLOC_MAX_POINTS) return GAL_ERR_TOO_LARGE;       // more partial sums than the array holds

    int prev = -1;
    cudaError_t e = cudaGetDevice(&prev);
    if (e != cudaSuccess) return noalloc_fail(e);
    if (prev != device && (e = cudaSetDevice(device)) != cudaSuccess) return noalloc_fail(e);
    struct Restore { int prev, dev; ~Restore() { if (prev != dev) cudaSetDevice(prev); } } restore{prev, device};

    cudaStream_t st = (cudaStream_t)stream;
    if (M == 0) {                                            // chi2 of no points
        if ((e = cudaMemsetAsync(chi2_out, 0, sizeof(double), st)) != cudaSuccess) return noalloc_fail(e);
        return GAL_OK;
    }
    unsigned char* scratch = nullptr;
    const int rc = noalloc_scratch_address(device, &scratch);
    if (rc) return rc;

    HankelParams h;
    h.I = I; h.nr = nr; h.Rmin = Rmin; h.dR = dR; h.inc_cos = std::cos(inc);
    h.cos_PA = std::cos(PA); h.sin_PA = std::sin(PA);         // PAPER.md:662-670, offsets kept in turns
    h.dRA_turns = dRA * h.cos_PA - dDec * h.sin_PA;
    h.dDec_turns = dRA * h.sin_PA + dDec * h.cos_PA;
    h.has_phase = !(h.dRA_turns == 0.0 && h.dDec_turns == 0.0);

    // the ticket must start at zero whatever the last call left behind
    if ((e = cudaMemsetAsync(scratch, 0, sizeof(unsigned int), st)) != cudaSuccess) return noalloc_fail(e);
    const unsigned tiles = (unsigned)((M + NOALLOC_TILE - 1) / NOALLOC_TILE);
    hankel_chi2_noalloc_kernel<<<tiles, NOALLOC_WARPS * 32, 0, st>>>(h, u, v, re_obs, im_obs, w, (long long)M, scratch,
                                                                     chi2_out);
    if ((e = cudaGetLastError()) != cudaSuccess) return noalloc_fail(e);
    return GAL_OK;
}

}  // extern "C"
