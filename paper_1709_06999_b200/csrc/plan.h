// plan.h — the plan object and the launcher interface between the C ABI (galario_b200.cu) and the per-precision
// kernel translation units (fft_f64.cu, fft_f32.cu, sample_f64.cu, sample_f32.cu).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <cstdlib>
#include <map>
#include <set>
#include <vector>

#include "../../include/galario_b200.h"
#include "types.h"

struct gal_plan {
    int nxy = 0, batch = 0, bits = 0, device = 0;
    int sm_count = 148;
    void* spec = nullptr;            // NodePair<T>[batch][nxy/2+1][nxy]: the sampled spectrum (column pairs)
    void* work = nullptr;            // cx<T>[batch][nxy/2+1][nxy]: row-pass output
    void* tw = nullptr;              // cx<T>[nxy]
    double* partials = nullptr;      // [batch][max_gx]
    unsigned int* tickets = nullptr; // [batch + 1]
    unsigned long long* oob = nullptr;   // call_state[0]; the uv extent follows it
    int* ext = nullptr;                  // {kumax, rmin, rmax} of the current call (device)
    int* ext_full = nullptr;             // constant {nxy/2, 0, nxy-1}: no pruning
    const int* cur_ext = nullptr;        // extent the current call's transform is pruned to (device); also selects the layout
    // Per-call device state [oob (8 B) | ext (12 B) | done ticket (4 B) | pad], two copies used alternately:
    // the sampling kernel of call k re-arms the copy call k+1 will use, so no reset operation sits between
    // two calls on the stream (an explicit copy from call_init is only needed when that did not happen).
    void* call_state = nullptr;          // 2 x 32 B
    void* call_init = nullptr;
    int cur = 0;                         // copy used by the most recent call
    bool next_armed = false;             // the other copy has been / will be re-armed by that call's sampler
    int prune_mode = 1;                  // 0 never, 1 auto, 2 always
    // tuning options (gal_plan_set_option; the defaults are the measured optimum on B200)
    int batch_chunk = 0;                 // GAL_OPT_BATCH_CHUNK: channels per chunk of a batched call (0: all in one chunk; galario_b200.cu batch_chunk)
    int row_mode = -1;                   // GAL_OPT_ROW_MODE, nxy 1024..4096: -1 per-size default, 0 plain row pass, 1 register-untangle kernel with plain loads, 2 its persistent TMA form, 3 one row per CTA
    int batch_conc = 12;                 // GAL_OPT_BATCH_CONC: channels in flight in the batched sampler
    double row_pf = 1.0;                 // GAL_OPT_ROW_PREFETCH: scale of the L2 prefetch distance of the FFT passes (0 = off)
    bool row_x2_one_cta = false;         // GAL_OPT_ROW_X2_ONE_CTA: nxy = 16384, one CTA per row instead of a cluster of two
    bool last_pruned = false;            // did the most recent call compute a uv extent?
    // bound uv set (gal_plan_bind_uv): addresses, size, the rotation-invariant radius, and the extent derived
    // from it for the pixel size seen last (device copy used by the FFT passes and checked by the sampler)
    const void* b_u = nullptr; const void* b_v = nullptr;
    int64_t b_M = 0; int b_C = 0;
    double b_rmax = 0.0, b_dxy = 0.0;
    int b_ext[3] = {0, 0, 0};
    int* b_ext_dev = nullptr;            // [4]
    unsigned long long* b_r2 = nullptr;  // [1] scratch of the radius kernel
    bool last_bound = false;             // the most recent call used the bound extent
    // bound observation set (gal_plan_bind_obs): the caller's five arrays (identity of the binding) and the plan's
    // private copy of them, sorted along a space-filling curve of the uv plane (sort.cuh); o_buf = [5][C][M]
    const void* o_src[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};
    int64_t o_M = 0; int o_C = 0;
    void* o_buf = nullptr; size_t o_bytes = 0;
    bool last_obs = false;               // the most recent call sampled the private copy
    // set (from the device, plain store to mapped host memory) by a sampler that found a point outside the extent
    // of a bound uv set: the promise was broken; the next call returns GAL_ERR_BINDING_VIOLATED
    unsigned int* viol_host = nullptr; unsigned int* viol_dev = nullptr;
    // viol_host[1] = extent hint, written by the last CTA of every sampling launch: 1 = that call's transform covered
    // the whole half plane, 2 = it was pruned.  The host reads it WITHOUT synchronising when it picks the row-pass
    // variant of the next call (a stale value costs time, never correctness): row_small = "expect a pruned extent".
    bool row_small = false;
    // Speculative extent (automatic pruning mode, one image per call, unbound uv, nxy 2048 / 4096): instead of a
    // uv-extent kernel in front of every call, the transform is pruned to the extent the previous call's sampler
    // derived from the largest baseline length of its points (rotation-invariant); the sampler verifies every point
    // against it and derives the extent for the next call; if a point lay outside, ONE conditional kernel (redo.cuh:
    // it leaves at once unless the device flag `redo` is set) repeats transform and sampling on the new extent.
    // No host synchronisation, results unchanged.
    // spec_state (device, 128 B): [0] u64 r2max | [8] int E[2][4] | [40] u32 redo | [44] int used_ext[3] | [64] u32 ctr[5] (redo.cuh)
    void* spec_state = nullptr;
    int spec_par = 0;                    // E[spec_par] is the extent the next speculative call transforms
    bool spec_valid = false;             // E[spec_par] has been (will have been, in stream order) written ...
    double spec_dxy = 0.0;               // ... for this pixel size
    cudaStream_t spec_stream = nullptr;  // ... on this stream
    int spec_mode = 0;                   // the launch being issued: 0 none, 1 derive only, 2 verify + derive
    bool spec_off = false;               // GAL_OPT_SPECULATE = 0
    double spec_min_bytes = 32e6;        // speculate only where the uv-extent pass would read at least this much (cfg 2, 16 MB: 42.0 against 44.5 us)
    bool last_spec = false;              // the most recent call speculated
    bool shared_spec = false;            // the call being issued samples ONE spectrum with every channel (gal_chi2_image_sets)
    int* spec_E(int par) const { return (int*)((char*)spec_state + 8 + 16 * par); }
    unsigned int* spec_redo() const { return (unsigned int*)((char*)spec_state + 40); }
    int* spec_used() const { return (int*)((char*)spec_state + 44); }
    unsigned int* spec_ctr() const { return (unsigned int*)((char*)spec_state + 64); }
    void* st_vis = nullptr; size_t st_vis_bytes = 0; // summed visibilities of a chi2 multi-source call
    std::set<const void*> smem_set;      // kernels whose dynamic shared-memory limit has been raised
    std::map<const void*, int> resident; // kernel -> CTAs resident on the whole GPU at once (occupancy x SM count)
    int max_gx = 0;
    size_t owned_bytes = 0;
    int last_cuda = 0;
    int64_t launches = 0;
    cudaStream_t last_stream = nullptr;
    // staging for the _host_ entry points (grown on demand)
    void* st_image = nullptr; size_t st_image_bytes = 0;
    void* st_pts = nullptr;   size_t st_pts_bytes = 0;
    void* st_out = nullptr;   size_t st_out_bytes = 0;
    double* st_chi2 = nullptr;
    // optional per-kernel timing (gal_plan_timing_enable): an event after every kernel of the recorded calls, each
    // tagged with what ended there (0 call start, 1 uv extent, 2 row pass, 3 column pass, 4 sampling)
    struct Mark { cudaEvent_t ev; int what; int call; };
    std::vector<Mark> tev;
    int t_max_calls = 0, t_calls = 0;
    bool t_on = false;               // the call being issued is recorded
    int tmark(int what, cudaStream_t st) {
        if (!t_on) return 0;
        Mark m; m.what = what; m.call = t_calls;
        cudaError_t e = cudaEventCreate(&m.ev);
        if (e == cudaSuccess) e = cudaEventRecord(m.ev, st);
        if (e != cudaSuccess) { last_cuda = (int)e; return -3; }
        tev.push_back(m);
        return 0;
    }
};

namespace galb {

#define GAL_CUDA(plan, call)                                   \
    do {                                                       \
        cudaError_t e__ = (call);                              \
        if (e__ != cudaSuccess) {                              \
            (plan)->last_cuda = (int)e__;                      \
            return e__ == cudaErrorMemoryAllocation ? GAL_ERR_ALLOC : GAL_ERR_CUDA; \
        }                                                      \
    } while (0)

struct DeviceGuard {
    int prev = -1;
    explicit DeviceGuard(int dev) { cudaGetDevice(&prev); if (prev != dev) cudaSetDevice(dev); else prev = -1; }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

template <typename K> inline int set_smem(gal_plan* p, K kernel, size_t bytes) {
    if (bytes > 48 * 1024 && !p->smem_set.count((const void*)kernel)) {
        GAL_CUDA(p, cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
        p->smem_set.insert((const void*)kernel);
    }
    return GAL_OK;
}

// CTAs of `kernel` resident on the GPU at once: the distance (in blocks) at which a CTA of an FFT pass prefetches
// into the L2 for a later one.  GAL_OPT_ROW_PREFETCH scales it (0 switches the prefetch off).
template <typename K> inline int resident_ctas(gal_plan* p, K kernel, int threads, size_t smem) {
    auto it = p->resident.find((const void*)kernel);
    if (it != p->resident.end()) return it->second;
    int per_sm = 1;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, threads, smem) != cudaSuccess || per_sm < 1) per_sm = 1;
    const int r = (int)(per_sm * p->sm_count * p->row_pf);
    p->resident[(const void*)kernel] = r;
    return r;
}

// Programmatic dependent launch: the kernels of one call form a chain on the stream; each is launched with
// programmatic stream serialisation so that its CTAs are placed and run their prologue while the kernel before
// drains, and each waits (`griddepcontrol.wait`, fft.cuh: pdl_wait) before it touches memory.
template <typename... KArgs, typename... Args>
inline cudaError_t launch_chain(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

// the same for a kernel whose CTAs form clusters of `cluster_x` along x (distributed shared memory)
template <typename... KArgs, typename... Args>
inline cudaError_t launch_chain_cluster(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, unsigned cluster_x, cudaStream_t st,
                                        Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute attr[2];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    attr[1].id = cudaLaunchAttributeClusterDimension;
    attr[1].val.clusterDim.x = cluster_x; attr[1].val.clusterDim.y = 1; attr[1].val.clusterDim.z = 1;
    cfg.attrs = attr; cfg.numAttrs = 2;
    return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

// ---- launchers, one explicit instantiation per precision (T = double in *_f64.cu, float in *_f32.cu) ----
// row pass + column pass of `batch` images (or of the swept profile) pruned to the device-resident extent `ext`
template <typename T> int fft2(gal_plan* p, const T* image, const SweepParams* sw, int batch, const int* ext, cudaStream_t st);
template <typename T> int launch_sweep(gal_plan* p, const SweepParams& sw, T* out, cudaStream_t st);
template <typename T> int launch_transpose(gal_plan* p, T* out, cudaStream_t st);
template <typename T> int launch_extent(gal_plan* p, int C, const CallScalars& cs, const T* u, const T* v, int64_t M, cudaStream_t st);
template <typename T> int launch_sample(gal_plan* p, int C, const CallScalars& cs, const T* u, const T* v, const T* re, const T* im,
                                        const T* w, int64_t M, T* vis, double* chi2_pc, double* chi2_tot, bool last, cudaStream_t st);
// conditional second pass of a speculative call: one persistent kernel (row pass, column pass, sampling behind grid
// barriers) on the extent E[spec_par ^ 1]; it does nothing unless the sampler before it raised the redo flag
template <typename T> int launch_redo(gal_plan* p, const T* image, const CallScalars& cs, const T* u, const T* v, const T* re,
                                      const T* im, const T* w, int64_t M, T* vis, double* chi2_pc, double* chi2_tot, cudaStream_t st);
template <typename T> int launch_sum_channels(gal_plan* p, const double* chi2_pc, int C, double* chi2_tot, cudaStream_t st);
// bind_obs: sort channel by channel, write the five sorted arrays to dst = [5][C][M]
template <typename T> int launch_bind_sort(gal_plan* p, const T* u, const T* v, const T* re, const T* im, const T* w, int64_t M,
                                           int C, double rmax, T* dst, cudaStream_t st);
template <typename T> int launch_hankel(gal_plan* p, const SweepParams& sw, const CallScalars& cs, const T* u, const T* v, const T* re,
                                        const T* im, const T* w, int64_t M, T* vis, double* chi2, cudaStream_t st);
template <typename T> int launch_sample_multi(gal_plan* p, const IndexScalars& ix, const PlacementSet& ps, const T* u, const T* v,
                                              const T* re, const T* im, const T* w, int64_t M, T* vis, bool write_vis,
                                              double* chi2, bool last, cudaStream_t st);
template <typename T> int launch_extent_radius(gal_plan* p, const T* u, const T* v, int64_t M, double du, cudaStream_t st);
template <typename T> int launch_uv_radius(gal_plan* p, const T* u, const T* v, long long total, cudaStream_t st);

}  // namespace galb
