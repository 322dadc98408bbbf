// triples_b200.cu -- C-ABI entry points of include/triples_b200.h and the host-side driver.
// No CPU fallback: every step of the hot path runs in the kernels of gemm_f64.cuh / gemm_f16split.cuh / reduce.cuh
// (plus ri_slices.cuh when the (vv|vo) slices are rebuilt from RI factors).
#include "../../include/triples_b200.h"

#include <cuda.h>
#include <cuda_runtime.h>

#include <algorithm>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <map>
#include <mutex>
#include <string>
#include <vector>

#include "gemm_emu64.cuh"
#include "gemm_f16split.cuh"
#include "gemm_f64.cuh"
#include "plan.h"
#include "prepare.cuh"
#include "probe.cuh"
#include "reduce.cuh"
#include "ri_slices.cuh"

// Scratch memory of triples_energy_noalloc: part of this library's device image, so a caller that cannot allocate
// device memory still has somewhere for the repacked operands, the U buffers and the job tables to live.  One copy per
// GPU that loads the image, held until the process exits.  In HOST code this name is only the host-side handle of
// the symbol, never a device address: the address a kernel may use comes from cudaGetSymbolAddress
// (noalloc_scratch below).
static __device__ __align__(256) unsigned char g_noalloc_scratch[TRIPLES_NOALLOC_SCRATCH_BYTES];

namespace {

using namespace tb;

thread_local std::string g_err;
constexpr int kProfSlots = 16;
thread_local double g_prof[kProfSlots];
thread_local bool g_prof_valid = false;
thread_local int g_profiling = 0;
thread_local long long g_launches = 0;   // kernels launched by the calling thread's last compute call

int fail(int code, const char* fmt, ...) {
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    g_err = buf;
    return code;
}

#define CU_TRY(expr)                                                                                  \
    do {                                                                                              \
        cudaError_t _e = (expr);                                                                      \
        if (_e != cudaSuccess)                                                                        \
            return fail(TRIPLES_ECUDA, "%s failed: %s (%s:%d)", #expr, cudaGetErrorString(_e), __FILE__, __LINE__); \
    } while (0)

// ------------------------------------------------------------------------------------------ tensor maps
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

int get_encode_fn(EncodeTiledFn* fn) {
    static EncodeTiledFn cached = nullptr;
    static std::mutex mu;
    std::lock_guard<std::mutex> lk(mu);
    if (!cached) {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult qres;
        CU_TRY(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres));
        if (qres != cudaDriverEntryPointSuccess || !p) return fail(TRIPLES_ECUDA, "cuTensorMapEncodeTiled unavailable");
        cached = reinterpret_cast<EncodeTiledFn>(p);
    }
    *fn = cached;
    return TRIPLES_OK;
}

// 3-D map over a dense tensor: dims d0 (fastest) .. d2, strides in elements for d1, d2; 128-byte swizzle.
int make_map3(CUtensorMap* m, CUtensorMapDataType dt, size_t esz, const void* base, uint64_t d0, uint64_t d1,
              uint64_t d2, uint64_t s1, uint64_t s2, uint32_t b0, uint32_t b1, uint32_t b2) {
    EncodeTiledFn fn;
    if (int rc = get_encode_fn(&fn)) return rc;
    cuuint64_t dims[3] = {d0, d1, d2};
    cuuint64_t strides[2] = {s1 * esz, s2 * esz};
    cuuint32_t box[3] = {b0, b1, b2};
    cuuint32_t estr[3] = {1, 1, 1};
    CUresult r = fn(m, dt, 3, const_cast<void*>(base), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                    CU_TENSOR_MAP_SWIZZLE_128B, dt == CU_TENSOR_MAP_DATA_TYPE_UINT32 ? CU_TENSOR_MAP_L2_PROMOTION_L2_128B : CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS)
        return fail(TRIPLES_ECUDA, "cuTensorMapEncodeTiled failed (%d) dims=%llu,%llu,%llu box=%u,%u,%u", (int)r,
                    (unsigned long long)d0, (unsigned long long)d1, (unsigned long long)d2, b0, b1, b2);
    return TRIPLES_OK;
}

// ------------------------------------------------------------------------------------------ device checks
int check_device() {
    int dev = 0;
    CU_TRY(cudaGetDevice(&dev));
    int major = 0;
    CU_TRY(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
    if (major != 10) return fail(TRIPLES_EARCH, "device %d has compute capability %d.x; this library is sm_100a only", dev, major);
    return TRIPLES_OK;
}

bool misaligned(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15) != 0; }

// A "device" argument must be device (or managed) memory of the current device: a host pointer would otherwise
// surface as a sticky CUDA error from inside a kernel.
int check_device_ptr(const void* p, const char* what, int n) {
    cudaPointerAttributes at;
    cudaError_t e = cudaPointerGetAttributes(&at, p);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return fail(TRIPLES_EINVAL, "%s #%d: cudaPointerGetAttributes failed (%s)", what, n, cudaGetErrorString(e));
    }
    if (at.type != cudaMemoryTypeDevice && at.type != cudaMemoryTypeManaged)
        return fail(TRIPLES_EINVAL, "%s #%d is not a device pointer", what, n);
    int dev = 0;
    CU_TRY(cudaGetDevice(&dev));
    if (at.type == cudaMemoryTypeDevice && at.device != dev)
        return fail(TRIPLES_EINVAL, "%s #%d lives on device %d, the current device is %d", what, n, at.device, dev);
    return TRIPLES_OK;
}

// The copy stream of streamed runs (one per device and host thread; created on first use, never destroyed).
thread_local std::map<int, cudaStream_t> g_copy_streams;
int copy_stream(cudaStream_t* out) {
    int dev = 0;
    CU_TRY(cudaGetDevice(&dev));
    auto it = g_copy_streams.find(dev);
    if (it == g_copy_streams.end()) {
        cudaStream_t s;
        CU_TRY(cudaStreamCreateWithFlags(&s, cudaStreamNonBlocking));
        it = g_copy_streams.emplace(dev, s).first;
    }
    *out = it->second;
    return TRIPLES_OK;
}

// ------------------------------------------------------------------------------------------ event pool
struct EventPool {
    std::vector<cudaEvent_t> ev;
    size_t used = 0;
    int get(cudaEvent_t* e) {
        if (used == ev.size()) {
            cudaEvent_t n;
            CU_TRY(cudaEventCreate(&n));
            ev.push_back(n);
        }
        *e = ev[used++];
        return TRIPLES_OK;
    }
    void reset() { used = 0; }
};
// One pool per device and host thread (like the copy streams): an event belongs to the device that was current when
// it was created, and recording it on another device's stream fails with an invalid resource handle.
thread_local std::map<int, EventPool> g_event_pools;
EventPool& event_pool() {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) dev = -1;
    return g_event_pools[dev];
}

// ------------------------------------------------------------------------------------------ contraction launch
// cudaFuncSetAttribute is per device and cheap: set on every launch (no process-wide "done" flag to race on).
template <int WM, int WN, int NT, int STAGES>
int launch_gemm_f64(const GemmMaps& maps, const GemmJob* jobs, int njobs, const Plan& P, cudaStream_t st) {
    using C = GemmF64Cfg<WM, WN, NT, STAGES>;
    auto kern = gemm_f64_kernel<WM, WN, NT, STAGES>;
    CU_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM_BYTES));
    const long long items = (long long)P.mtiles * P.ntiles * njobs;
    if (items == 0) return TRIPLES_OK;
    const int grid = (int)std::min<long long>(items, kNumSM);     // persistent: one CTA per SM
    kern<<<grid, C::THREADS, C::SMEM_BYTES, st>>>(maps, jobs, njobs, P.v, P.vp, P.o, P.mtiles, P.ntiles);
    CU_TRY(cudaGetLastError());
    ++g_launches;
    return TRIPLES_OK;
}

// word of the scales block that pack_xk_kernel sets when a scaled (vv|vo) element exceeds its class bound
constexpr int kOverflowWord = 14;

struct Operands {   // device pointers of the repacked operands (workspace) for one precision
    void *x, *xt, *ot, *t2;
    void *t2k, *t2kt;   // mixed path only
    float* scales;      // mixed path only: 2^sg, 2^st, 2^-(sg+st) (prepare.cuh scales_kernel), then two uint maxima
    double* stage;      // FP64 staging slices (mixed streamed / RI)
    double *bt, *bo;    // RI mode: repacked factors
};

struct Maps {   // tensor maps of the contraction kernel of the plan's precision
    GemmMaps f64;
    SplitMaps split;
    EmuMaps emu;
    RiMaps ri;
};

int build_maps_f64(const Plan& P, const Operands& op, GemmMaps* maps) {
    const uint64_t o = P.o, v = P.v, vp = P.vp, opp = P.op, N = v * vp, ns = P.nslots;
    const CUtensorMapDataType dt = CU_TENSOR_MAP_DATA_TYPE_FLOAT64;
    int rc;
    if ((rc = make_map3(&maps->t2a, dt, 8, op.t2, v, v, o * o, vp, v * vp, 16, P.BM, 1))) return rc;
    if ((rc = make_map3(&maps->ota, dt, 8, op.ot, o, v, o * o, opp, v * opp, 16, P.BM, 1))) return rc;
    if ((rc = make_map3(&maps->x, dt, 8, op.x, N, v, ns, N, v * N, 16, 16, 1))) return rc;
    if ((rc = make_map3(&maps->xt, dt, 8, op.xt, N, v, ns, N, v * N, 16, 16, 1))) return rc;
    if ((rc = make_map3(&maps->t2bq, dt, 8, op.t2, N, o, o, N, o * N, 16, 16, 1))) return rc;
    if ((rc = make_map3(&maps->t2br, dt, 8, op.t2, N, o, o, N, o * N, 16, 1, 16))) return rc;
    return TRIPLES_OK;
}

// packed operands: 4-byte words (FP16 pairs), 32 words = one 128-byte row per K chunk
int build_maps_split(const Plan& P, const Operands& op, SplitMaps* maps) {
    const uint64_t o = P.o, v = P.v, vk = P.vk, ok = P.ok, NR = (uint64_t)P.v * P.vp, ns = P.nslots;
    const CUtensorMapDataType dt = CU_TENSOR_MAP_DATA_TYPE_UINT32;
    int rc;
    if ((rc = make_map3(&maps->xk, dt, 4, op.x, vk, NR, ns, vk, NR * vk, FS_BK, FS_BM, 1))) return rc;
    if ((rc = make_map3(&maps->xkt, dt, 4, op.xt, vk, NR, ns, vk, NR * vk, FS_BK, FS_BM, 1))) return rc;
    if ((rc = make_map3(&maps->t2k, dt, 4, op.t2k, ok, NR, o, ok, NR * ok, FS_BK, FS_BM, 1))) return rc;
    if ((rc = make_map3(&maps->t2kt, dt, 4, op.t2kt, ok, NR, o, ok, NR * ok, FS_BK, FS_BM, 1))) return rc;
    if ((rc = make_map3(&maps->t2a, dt, 4, op.t2, vk, v, o * o, vk, v * vk, FS_BK, P.tf_npad, 1))) return rc;
    if ((rc = make_map3(&maps->ota, dt, 4, op.ot, ok, v, o * o, ok, v * ok, FS_BK, P.tf_npad, 1))) return rc;
    return TRIPLES_OK;
}

// emulated-FP64 operands: 64 words (two 128-byte rows of digits) per K chunk; a box is one of the two rows
int build_maps_emu(const Plan& P, const Operands& op, EmuMaps* maps) {
    const uint64_t o = P.o, v = P.v, vk = P.vk, ok = P.ok, NR = (uint64_t)P.v * P.vp, ns = P.nslots;
    const CUtensorMapDataType dt = CU_TENSOR_MAP_DATA_TYPE_UINT32;
    int rc;
    if ((rc = make_map3(&maps->xk, dt, 4, op.x, vk, NR, ns, vk, NR * vk, 32, EM_BM, 1))) return rc;
    if ((rc = make_map3(&maps->xkt, dt, 4, op.xt, vk, NR, ns, vk, NR * vk, 32, EM_BM, 1))) return rc;
    if ((rc = make_map3(&maps->t2k, dt, 4, op.t2k, ok, NR, o, ok, NR * ok, 32, EM_BM, 1))) return rc;
    if ((rc = make_map3(&maps->t2kt, dt, 4, op.t2kt, ok, NR, o, ok, NR * ok, 32, EM_BM, 1))) return rc;
    if ((rc = make_map3(&maps->t2a, dt, 4, op.t2, vk, v, o * o, vk, v * vk, 32, P.tf_npad, 1))) return rc;
    if ((rc = make_map3(&maps->ota, dt, 4, op.ot, ok, v, o * o, ok, v * ok, 32, P.tf_npad, 1))) return rc;
    return TRIPLES_OK;
}

int build_maps_ri(const Plan& P, const Operands& op, RiMaps* maps) {
    const uint64_t v = P.v, vp = P.vp, o = P.o, na = P.naux, nap = P.nauxp;
    const CUtensorMapDataType dt = CU_TENSOR_MAP_DATA_TYPE_FLOAT64;
    int rc;
    if ((rc = make_map3(&maps->bt, dt, 8, op.bt, na, v * v, 1, nap, v * v * nap, 16, P.ri_BM, 1))) return rc;
    if ((rc = make_map3(&maps->bo, dt, 8, op.bo, vp, na, o, vp, na * vp, 16, 16, 1))) return rc;
    return TRIPLES_OK;
}

int build_maps(const Plan& P, const Operands& op, Maps* maps) {
    if (P.mode == SLICES_RI)
        if (int rc = build_maps_ri(P, op, &maps->ri)) return rc;
    if (P.prec == TRIPLES_EMU64) return build_maps_emu(P, op, &maps->emu);
    return P.prec == TRIPLES_FP64 ? build_maps_f64(P, op, &maps->f64) : build_maps_split(P, op, &maps->split);
}

// co-resident CTA pairs of a tcgen05 contraction kernel, per (kernel, device, shared-memory request)
template <typename K>
int max_pair_clusters(K kern, int which, cudaLaunchConfig_t cfg, int cs, int* out) {
    static std::mutex mu;
    static std::map<std::pair<int, size_t>, int> cache;
    int dev = 0;
    CU_TRY(cudaGetDevice(&dev));
    std::lock_guard<std::mutex> lk(mu);
    const auto key = std::make_pair(dev * 8 + which, cfg.dynamicSmemBytes);
    auto it = cache.find(key);
    if (it == cache.end()) {
        cfg.gridDim = dim3(kNumSM / cs * cs);
        int n = 0;
        CU_TRY(cudaOccupancyMaxActiveClusters(&n, kern, &cfg));
        if (n < 1) return fail(TRIPLES_ECUDA, "no CTA pair of the tcgen05 contraction fits the device");
        it = cache.emplace(key, std::min(n, kNumSM / cs)).first;
    }
    *out = it->second;
    return TRIPLES_OK;
}

int launch_gemm_split(const SplitMaps& maps, const GemmJob* jobs, int njobs, const Plan& P, const float* scales,
                      cudaStream_t st) {
    CU_TRY(cudaFuncSetAttribute(gemm_f16split_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, FS_SMEM_LIMIT));
    const int cs = P.tf_cs;
    if (njobs > FS_MAX_JOBS) return fail(TRIPLES_EINVAL, "internal: %d contraction jobs in one launch (max %d)", njobs, FS_MAX_JOBS);
    const long long items = (long long)njobs * ((P.tf_mtiles + cs - 1) / cs) * P.tf_ntiles;   // per cluster
    if (items == 0) return TRIPLES_OK;
    cudaLaunchConfig_t cfg = {};
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = cs; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.blockDim = dim3(FS_THREADS);
    cfg.dynamicSmemBytes = fs_smem_bytes(P.tf_npad);
    cfg.stream = st;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    int max_clusters = 0;
    if (int rc = max_pair_clusters(gemm_f16split_kernel, 0, cfg, cs, &max_clusters)) return rc;
    cfg.gridDim = dim3((unsigned)(std::min<long long>(items, max_clusters) * cs));
    CU_TRY(cudaLaunchKernelEx(&cfg, gemm_f16split_kernel, maps, jobs, njobs, P.v, P.vp, P.o, P.tf_mtiles, P.tf_ntiles,
                              P.tf_bn, P.tf_npad, scales));
    ++g_launches;
    return TRIPLES_OK;
}

template <int BN>
int launch_gemm_emu_t(const EmuMaps& maps, const GemmJob* jobs, int njobs, const Plan& P, const float* scales,
                      cudaStream_t st) {
    auto kern = gemm_emu64_kernel<BN>;
    CU_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, em_smem_bytes(BN)));
    const int cs = P.tf_cs;
    if (njobs > EM_MAX_JOBS) return fail(TRIPLES_EINVAL, "internal: %d contraction jobs in one launch (max %d)", njobs, EM_MAX_JOBS);
    const long long items = (long long)njobs * ((P.tf_mtiles + cs - 1) / cs) * P.tf_ntiles;
    if (items == 0) return TRIPLES_OK;
    cudaLaunchConfig_t cfg = {};
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = cs; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.blockDim = dim3(EM_THREADS);
    cfg.dynamicSmemBytes = em_smem_bytes(BN);
    cfg.stream = st;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    int max_clusters = 0;
    if (int rc = max_pair_clusters(kern, 1 + BN / 16, cfg, cs, &max_clusters)) return rc;
    cfg.gridDim = dim3((unsigned)(std::min<long long>(items, max_clusters) * cs));
    CU_TRY(cudaLaunchKernelEx(&cfg, kern, maps, jobs, njobs, P.v, P.vp, P.o, P.tf_mtiles, P.tf_ntiles, scales));
    ++g_launches;
    return TRIPLES_OK;
}

int launch_gemm_emu(const EmuMaps& maps, const GemmJob* jobs, int njobs, const Plan& P, const float* scales,
                    cudaStream_t st) {
    switch (P.tf_bn) {
        case 80: return launch_gemm_emu_t<80>(maps, jobs, njobs, P, scales, st);
        case 64: return launch_gemm_emu_t<64>(maps, jobs, njobs, P, scales, st);
        default: return launch_gemm_emu_t<48>(maps, jobs, njobs, P, scales, st);
    }
}

int launch_gemm(const Plan& P, const Maps& maps, const Operands& op, const GemmJob* jobs, int njobs, cudaStream_t st) {
    if (P.prec == TRIPLES_MIXED) return launch_gemm_split(maps.split, jobs, njobs, P, op.scales, st);
    if (P.prec == TRIPLES_EMU64) return launch_gemm_emu(maps.emu, jobs, njobs, P, op.scales, st);
    switch (P.cfg) {
        case CFG_M120_N128: return launch_gemm_f64<3, 4, 4, 4>(maps.f64, jobs, njobs, P, st);
        case CFG_M80_N192: return launch_gemm_f64<2, 6, 4, 4>(maps.f64, jobs, njobs, P, st);
        default: return launch_gemm_f64<1, 8, 4, 4>(maps.f64, jobs, njobs, P, st);
    }
}

template <int WM, int WN, int NT, int STAGES>
int launch_ri_t(const RiMaps& maps, const int2* loads, int nloads, const Plan& P, double* X, cudaStream_t st) {
    using C = GemmF64Cfg<WM, WN, NT, STAGES>;
    auto kern = ri_slice_kernel<WM, WN, NT, STAGES>;
    CU_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM_BYTES));
    const long long items = (long long)P.ri_mtiles * P.ri_ntiles * nloads;
    if (items == 0) return TRIPLES_OK;
    const int grid = (int)std::min<long long>(items, kNumSM);
    kern<<<grid, C::THREADS, C::SMEM_BYTES, st>>>(maps, loads, nloads, P.v, P.vp, P.naux, P.ri_mtiles, P.ri_ntiles, X,
                                                  (size_t)P.v * P.v * P.vp);
    CU_TRY(cudaGetLastError());
    ++g_launches;
    return TRIPLES_OK;
}

// X_r of every load, FP64 natural order, into slot `loads[n].y` of X
int launch_ri(const Plan& P, const Maps& maps, const int2* loads, int nloads, double* X, cudaStream_t st) {
    switch (P.ri_cfg) {
        case CFG_M120_N128: return launch_ri_t<3, 4, 4, 4>(maps.ri, loads, nloads, P, X, st);
        case CFG_M80_N192: return launch_ri_t<2, 6, 4, 4>(maps.ri, loads, nloads, P, X, st);
        default: return launch_ri_t<1, 8, 4, 4>(maps.ri, loads, nloads, P, X, st);
    }
}

// ------------------------------------------------------------------------------------------ prepare (S0)
struct Inputs {
    const double *eps_o, *eps_v, *t1, *t2, *ovoo, *ovov;
};

// Where the (vv|vo) slices come from (plan.h SliceMode)
struct Source {
    int mode = SLICES_RESIDENT;
    const double* vvvo = nullptr;        // resident: device [a][b][c][k]
    const double* vovv_host = nullptr;   // streamed: host [k][a][b][c] = (ab|ck)
    double absmax = 0.0;                 // streamed, mixed: largest |(ab|ck)| if the caller knows it (else scanned)
    const double* B = nullptr;           // RI: device [naux][n][n], n = o + v, occupied orbitals first
};

struct RunOpts { int shard = 0, nshards = 1; };

// XT = X with every (b,c) plane transposed, for `nslices` consecutive slices (v planes each); gridDim.z <= 65535
int transpose_slices(const Plan& P, const double* X, double* XT, int nslices, cudaStream_t st) {
    const size_t plane = (size_t)P.v * P.vp;
    for (long long z0 = 0, nz = (long long)nslices * P.v; z0 < nz; z0 += 65535) {
        dim3 grid((P.v + 31) / 32, (P.v + 31) / 32, (unsigned)std::min<long long>(65535, nz - z0));
        transpose_planes_kernel<double><<<grid, 256, 0, st>>>(X + (size_t)z0 * plane, P.v, P.vp, XT + (size_t)z0 * plane);
        CU_TRY(cudaGetLastError());
        ++g_launches;
    }
    return TRIPLES_OK;
}
int transpose_slice(const Plan& P, const double* X, double* XT, cudaStream_t st) { return transpose_slices(P, X, XT, 1, st); }

// src viewed as [d][s]: the resident vvvo (ro = o, slot = r) or one FP64 slice (ro = 1) -> packed XK / XKT slots
int pack_xk(const Plan& P, const double* src, int ro, int sp, int slot0, const Operands& op, cudaStream_t st) {
    auto kern = P.prec == TRIPLES_EMU64 ? pack_xk_kernel<1> : pack_xk_kernel<0>;
    CU_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, PKX_SMEM));
    const size_t S = (size_t)P.v * P.v * ro;
    dim3 grid((unsigned)((S + PKX_SPAN - 1) / PKX_SPAN), P.kchunks_v);
    kern<<<grid, 256, PKX_SMEM, st>>>(src, P.v, P.vp, P.vk, ro, sp, slot0, (uint32_t*)op.x, (uint32_t*)op.xt, op.scales,
                                      reinterpret_cast<unsigned int*>(op.scales) + kOverflowWord);
    CU_TRY(cudaGetLastError());
    ++g_launches;
    return TRIPLES_OK;
}

// The small operands (t2, ovoo) and, for a resident vvvo, all slices.  Mixed path: the two power-of-two scales first.
int run_prepare(const Plan& P, const Inputs& in, const Source& src, const Operands& op, cudaStream_t st,
                cudaStream_t copy_st) {
    const int o = P.o, v = P.v;
    if (P.vp != v) {   // pad rows / columns c = v stay zero (never written by the repack kernels)
        CU_TRY(cudaMemsetAsync(op.x, 0, P.n_x * P.osz, st));
        CU_TRY(cudaMemsetAsync(op.xt, 0, P.n_x * P.osz, st));
        if (P.prec == TRIPLES_FP64) CU_TRY(cudaMemsetAsync(op.t2, 0, P.n_t2 * 8, st));
    }
    if (P.prec == TRIPLES_FP64) {
        if (P.op != o) CU_TRY(cudaMemsetAsync(op.ot, 0, P.n_ot * 8, st));
        if (src.mode == SLICES_RESIDENT) {
            int RB = 128;
            while ((size_t)RB * (o + 1) * 8 > 64 * 1024 && RB > 1) RB /= 2;
            const size_t R = (size_t)v * v * v;
            const size_t smem = (size_t)RB * (o + 1) * 8;
            auto kern = pack_x_kernel<double>;
            CU_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024));
            kern<<<(unsigned)((R + RB - 1) / RB), 256, smem, st>>>(src.vvvo, v, P.vp, o, RB, (double*)op.x);
            CU_TRY(cudaGetLastError());
            ++g_launches;
            if (int rc = transpose_slices(P, (const double*)op.x, (double*)op.xt, o, st)) return rc;
        }
        pack_ot_kernel<double><<<kNumSM * 4, 256, 0, st>>>(in.ovoo, v, o, P.op, (double*)op.ot);
        CU_TRY(cudaGetLastError());
        ++g_launches;
        pack_t2_kernel<double><<<kNumSM * 8, 256, 0, st>>>(in.t2, (size_t)o * o * v, v, P.vp, (double*)op.t2);
        CU_TRY(cudaGetLastError());
        ++g_launches;
        return TRIPLES_OK;
    }
    // ---- packed paths (mixed: FP16 split; emulated FP64: base-256 digits)
    const bool emu = P.prec == TRIPLES_EMU64;
    if (P.vp != v) {
        CU_TRY(cudaMemsetAsync(op.t2k, 0, P.n_t2k * 4, st));
        CU_TRY(cudaMemsetAsync(op.t2kt, 0, P.n_t2k * 4, st));
    }
    {   // power-of-two scales of the two tensor classes: maxima as float bit patterns, integrals | t2
        unsigned int* mx = reinterpret_cast<unsigned int*>(op.scales + 4);
        CU_TRY(cudaMemsetAsync(mx, 0, 48, st));     // two maxima, (RI) two factor norms at scales + 8, overflow flag
        const size_t nv3 = (size_t)v * v * v;
        if (src.mode == SLICES_RESIDENT) {
            absmax_kernel<<<kNumSM * 8, 256, 0, st>>>(src.vvvo, nv3 * o, mx);
            ++g_launches;
        } else if (src.mode == SLICES_STREAMED) {
            if (src.absmax > 0.0) {
                const float m = (float)src.absmax;      // pageable source: staged before the call returns
                CU_TRY(cudaMemcpyAsync(mx, &m, 4, cudaMemcpyHostToDevice, st));
            } else {   // one pass over the host tensor (two staging slices, copies overlap the scans)
                cudaEvent_t scanned[2] = {nullptr, nullptr}, landed = nullptr;
                for (int r = 0; r < o; ++r) {
                    double* stg = op.stage + (size_t)(r & 1) * nv3;
                    if (scanned[r & 1]) CU_TRY(cudaStreamWaitEvent(copy_st, scanned[r & 1], 0));
                    CU_TRY(cudaMemcpyAsync(stg, src.vovv_host + (size_t)r * nv3, nv3 * 8, cudaMemcpyHostToDevice, copy_st));
                    if (int rc = event_pool().get(&landed)) return rc;
                    CU_TRY(cudaEventRecord(landed, copy_st));
                    CU_TRY(cudaStreamWaitEvent(st, landed, 0));
                    absmax_kernel<<<kNumSM * 8, 256, 0, st>>>(stg, nv3, mx);
                    ++g_launches;
                    if (int rc = event_pool().get(&scanned[r & 1])) return rc;
                    CU_TRY(cudaEventRecord(scanned[r & 1], st));
                }
            }
        } else {   // RI: Cauchy-Schwarz bound |(ab|cr)| <= |B[:,a,b]| |B[:,c,r]| over the factor columns
            ri_bound_kernel<<<kNumSM * 4, 256, 0, st>>>(src.B, o, v, P.naux, op.scales + 8);
            ri_bound_fold_kernel<<<1, 32, 0, st>>>(op.scales + 8, mx);
            g_launches += 2;
        }
        absmax_kernel<<<kNumSM, 256, 0, st>>>(in.ovoo, (size_t)o * v * o * o, mx);
        absmax_kernel<<<kNumSM * 2, 256, 0, st>>>(in.t2, (size_t)o * o * v * v, mx + 1);
        scales_kernel<<<1, 32, 0, st>>>(mx, op.scales);
        CU_TRY(cudaGetLastError());
        g_launches += 3;
    }
    if (src.mode == SLICES_RESIDENT)
        if (int rc = pack_xk(P, src.vvvo, o, v, 0, op, st)) return rc;
    {
        dim3 grid(o * v, (v + 63) / 64, (o + 63) / 64);
        (emu ? pack_t2k_kernel<1> : pack_t2k_kernel<0>)<<<grid, 256, 0, st>>>(in.t2, v, P.vp, o, P.ok, (uint32_t*)op.t2k,
                                                                               (uint32_t*)op.t2kt, op.scales);
        CU_TRY(cudaGetLastError());
        ++g_launches;
    }
    (emu ? pack_ota_kernel<1> : pack_ota_kernel<0>)<<<kNumSM * 4, 256, 0, st>>>(in.ovoo, v, o, P.ok, (uint32_t*)op.ot, op.scales);
    CU_TRY(cudaGetLastError());
    ++g_launches;
    (emu ? pack_t2a_kernel<1> : pack_t2a_kernel<0>)<<<kNumSM * 8, 256, 0, st>>>(in.t2, (size_t)o * o * v, v, P.vk,
                                                                                 (uint32_t*)op.t2, op.scales);
    CU_TRY(cudaGetLastError());
    ++g_launches;
    return TRIPLES_OK;
}

Operands carve_operands(const Plan& P, uint8_t* ws) {
    Operands op{};
    op.x = ws + P.off_x; op.xt = ws + P.off_xt; op.ot = ws + P.off_ot; op.t2 = ws + P.off_t2;
    if (P.prec != TRIPLES_FP64) {
        op.t2k = ws + P.off_t2k; op.t2kt = ws + P.off_t2kt;
        op.scales = reinterpret_cast<float*>(ws + P.off_result + 64);   // the result block has 256 bytes, 24 used
    }
    if (P.nstage) op.stage = reinterpret_cast<double*>(ws + P.off_stage);
    if (P.mode == SLICES_RI) {
        op.bt = reinterpret_cast<double*>(ws + P.off_bt);
        op.bo = reinterpret_cast<double*>(ws + P.off_bo);
    }
    return op;
}

// ------------------------------------------------------------------------------------------ core driver
// Runs prepare + all batches of this shard for `trip` (restricted triplets, index = row of e_trip to write) and
// leaves the weighted per-triplet energies in e_trip (device, 3 doubles per row; rows of i=j=k triplets and of
// triplets of other shards are zero).
template <typename TS>
int run_batches(const Plan& P, const Inputs& in, const Source& src, uint8_t* ws, cudaStream_t st,
                const std::vector<Triplet>& trip, double* e_trip, size_t e_trip_rows, const RunOpts& opt) {
    const int o = P.o, v = P.v;
    Operands op = carve_operands(P, ws);
    const bool prof = g_profiling != 0;
    const bool streamed = P.mode == SLICES_STREAMED, ri = P.mode == SLICES_RI;
    event_pool().reset();

    // ---- batches, shard, slice cache and job tables (plan.h)
    BatchPlan B;
    build_batches(P, trip, B);
    select_shard(B, opt.shard, opt.nshards);
    if (P.mode != SLICES_RESIDENT && !build_slices(o, P.nslots, streamed, B))
        return fail(TRIPLES_EWORKSPACE, "slice cache of %d slots is too small for batches of window %d", P.nslots, P.win);
    const std::vector<Triplet>& work = B.work;
    const std::vector<size_t>& bstart = B.bstart;
    const std::vector<int>& gj_begin = B.jstart;
    const size_t nwork = work.size(), nbatch = bstart.size() - 1;

    cudaStream_t cs = nullptr;
    if (streamed) {
        if (int rc = copy_stream(&cs)) return rc;
        cudaEvent_t ev_start;       // the copy stream may not touch the workspace before earlier work on `st` is done
        if (int rc = event_pool().get(&ev_start)) return rc;
        CU_TRY(cudaEventRecord(ev_start, st));
        CU_TRY(cudaStreamWaitEvent(cs, ev_start, 0));
    }
    cudaEvent_t ev_p0 = nullptr, ev_p1 = nullptr;
    if (prof) {
        if (int rc = event_pool().get(&ev_p0)) return rc;
        if (int rc = event_pool().get(&ev_p1)) return rc;
        CU_TRY(cudaEventRecord(ev_p0, st));
    }
    if (int rc = run_prepare(P, in, src, op, st, cs)) return rc;
    if (ri) {
        dim3 g1((unsigned)(((size_t)v * v + 31) / 32), (P.nauxp + 31) / 32);
        ri_pack_bt_kernel<<<g1, 256, 0, st>>>(src.B, o, v, P.naux, P.nauxp, op.bt);
        ri_pack_bo_kernel<<<kNumSM * 8, 256, 0, st>>>(src.B, o, v, P.naux, P.vp, op.bo);
        CU_TRY(cudaGetLastError());
        g_launches += 2;
    }
    if (prof) CU_TRY(cudaEventRecord(ev_p1, st));
    cudaEvent_t ev_prepared = nullptr;
    if (streamed) {   // pad memsets / scale scan precede the first slice copy
        if (int rc = event_pool().get(&ev_prepared)) return rc;
        CU_TRY(cudaEventRecord(ev_prepared, st));
        CU_TRY(cudaStreamWaitEvent(cs, ev_prepared, 0));
    }

    Maps maps;
    if (int rc = build_maps(P, op, &maps)) return rc;

    std::vector<Orbit> orbits;
    enumerate_orbits(v, orbits);
    const double distinct_u = B.distinct_u;
    TS* ubase = reinterpret_cast<TS*>(ws + P.off_u);
    std::vector<GemmJob> gj(B.jobs.size());
    for (size_t n = 0; n < gj.size(); ++n) {
        const JobDesc& d = B.jobs[n];
        TS* ub = ubase + (size_t)3 * d.slot * P.n_u;      // interleaved blocks of U1,U2,U3 of the slot (ulayout.cuh)
        gj[n] = {d.p, d.q, d.r, d.gstart, ub + (size_t)d.u * UBLK, d.u2 < 0 ? nullptr : ub + (size_t)d.u2 * UBLK,
                 d.gsize, d.xr, d.xq, 0};
    }
    std::vector<RedJob> rj(nwork);
    std::vector<FinJob> fj(nwork);
    for (size_t b = 0; b < nbatch; ++b)
        for (size_t n = bstart[b]; n < bstart[b + 1]; ++n) {
            const Triplet& t = work[n];
            const int slot = (int)(n - bstart[b]);
            rj[n] = {t.i, t.j, t.k, slot, ubase + (size_t)3 * slot * P.n_u, nullptr};
            fj[n] = {slot, (int)t.index, triplet_weight(t.i, t.j, t.k)};
        }
    GemmJob* d_gj = reinterpret_cast<GemmJob*>(ws + P.off_gjobs);
    RedJob* d_rj = reinterpret_cast<RedJob*>(ws + P.off_rjobs);
    double* d_side = reinterpret_cast<double*>(ws + P.off_side);
    static_assert(kRedWarps == RED_CONSUMER_WARPS, "plan.h and reduce.cuh disagree");
    CU_TRY(cudaFuncSetAttribute(reduce_kernel<TS>, cudaFuncAttributeMaxDynamicSharedMemorySize, RedCfg<TS>::SMEM_BYTES));
    FinJob* d_fj = reinterpret_cast<FinJob*>(ws + P.off_fjobs);
    uchar4* d_orb = reinterpret_cast<uchar4*>(ws + P.off_orb);
    double2* d_part = reinterpret_cast<double2*>(ws + P.off_part);
    int2* d_loads = reinterpret_cast<int2*>(ws + P.off_loads);
    if (!gj.empty()) CU_TRY(cudaMemcpyAsync(d_gj, gj.data(), gj.size() * sizeof(GemmJob), cudaMemcpyHostToDevice, st));
    if (nwork) {
        CU_TRY(cudaMemcpyAsync(d_rj, rj.data(), nwork * sizeof(RedJob), cudaMemcpyHostToDevice, st));
        CU_TRY(cudaMemcpyAsync(d_fj, fj.data(), nwork * sizeof(FinJob), cudaMemcpyHostToDevice, st));
    }
    // RI: the load table {r, slot}, followed by the same loads aimed at staging slice 0 (mixed path)
    std::vector<int2> ltab(2 * B.loads.size());
    for (size_t l = 0; l < B.loads.size(); ++l) {
        ltab[l] = make_int2(B.loads[l].r, B.loads[l].slot);
        ltab[B.loads.size() + l] = make_int2(B.loads[l].r, 0);
    }
    if (ri && !ltab.empty())
        CU_TRY(cudaMemcpyAsync(d_loads, ltab.data(), ltab.size() * sizeof(int2), cudaMemcpyHostToDevice, st));
    CU_TRY(cudaMemcpyAsync(d_orb, orbits.data(), orbits.size() * sizeof(Orbit), cudaMemcpyHostToDevice, st));
    CU_TRY(cudaMemsetAsync(e_trip, 0, e_trip_rows * 3 * sizeof(double), st));

    // ---- streamed slices: H2D copies on the copy stream, two batches ahead of the contraction that needs them
    const size_t nv3 = (size_t)v * v * v;
    std::vector<cudaEvent_t> ev_loaded(streamed ? nbatch : 0), ev_gemm(streamed ? nbatch : 0);
    double h2d_bytes = 0.0;
    auto stage_of = [&](size_t b, int li) { return op.stage + ((b & 1) * (size_t)(P.nstage / 2) + li) * nv3; };
    auto enqueue_copies = [&](size_t b) -> int {
        if (b >= nbatch) return TRIPLES_OK;
        if (b >= 2) CU_TRY(cudaStreamWaitEvent(cs, ev_gemm[b - 2], 0));     // frees the slots / staging half it reuses
        for (int l = B.lstart[b]; l < B.lstart[b + 1]; ++l) {
            const SliceLoad& ld = B.loads[l];
            const double* hsrc = src.vovv_host + (size_t)ld.r * nv3;
            if (P.prec == TRIPLES_FP64)      // the host slice [d][b][c] IS X_r: straight into its slot (c-pitch vp)
                CU_TRY(cudaMemcpy2DAsync((double*)op.x + (size_t)ld.slot * P.n_slice, (size_t)P.vp * 8, hsrc, (size_t)v * 8,
                                         (size_t)v * 8, (size_t)v * v, cudaMemcpyHostToDevice, cs));
            else
                CU_TRY(cudaMemcpyAsync(stage_of(b, l - B.lstart[b]), hsrc, nv3 * 8, cudaMemcpyHostToDevice, cs));
            h2d_bytes += (double)nv3 * 8;
        }
        if (int rc = event_pool().get(&ev_loaded[b])) return rc;
        CU_TRY(cudaEventRecord(ev_loaded[b], cs));
        return TRIPLES_OK;
    };
    if (streamed) {
        if (int rc = enqueue_copies(0)) return rc;
        if (int rc = enqueue_copies(1)) return rc;
    }

    // ---- batches: [slices ->] contraction -> fused reduction -> per-triplet finalize
    std::vector<cudaEvent_t> evs;
    for (size_t b = 0; b < nbatch; ++b) {
        const size_t n0 = bstart[b];
        const int cnt = (int)(bstart[b + 1] - n0);
        const int g0 = gj_begin[b], g1 = gj_begin[b + 1];
        cudaEvent_t e[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};
        if (prof) {
            for (int x = 0; x < 5; ++x) if (int rc = event_pool().get(&e[x])) return rc;
            CU_TRY(cudaEventRecord(e[4], st));
        }
        if (P.mode != SLICES_RESIDENT) {
            const int l0 = B.lstart[b], l1 = B.lstart[b + 1];
            if (streamed) CU_TRY(cudaStreamWaitEvent(st, ev_loaded[b], 0));
            if (ri && l1 > l0) {
                if (P.prec == TRIPLES_FP64) {
                    if (int rc = launch_ri(P, maps, d_loads + l0, l1 - l0, (double*)op.x, st)) return rc;
                } else {   // one FP64 staging slice: build, split-pack, next
                    for (int l = l0; l < l1; ++l) {
                        if (int rc = launch_ri(P, maps, d_loads + B.loads.size() + l, 1, op.stage, st)) return rc;
                        if (int rc = pack_xk(P, op.stage, 1, P.vp, B.loads[l].slot, op, st)) return rc;
                    }
                }
            }
            for (int l = l0; l < l1; ++l) {
                const SliceLoad& ld = B.loads[l];
                if (P.prec == TRIPLES_FP64) {
                    if (int rc = transpose_slice(P, (const double*)op.x + (size_t)ld.slot * P.n_slice,
                                                 (double*)op.xt + (size_t)ld.slot * P.n_slice, st)) return rc;
                } else if (streamed) {
                    if (int rc = pack_xk(P, stage_of(b, l - l0), 1, v, ld.slot, op, st)) return rc;
                }
            }
        }
        if (prof) CU_TRY(cudaEventRecord(e[0], st));
        if (int rc = launch_gemm(P, maps, op, d_gj + g0, g1 - g0, st)) return rc;
        if (prof) CU_TRY(cudaEventRecord(e[1], st));
        if (streamed) {
            if (int rc = event_pool().get(&ev_gemm[b])) return rc;
            CU_TRY(cudaEventRecord(ev_gemm[b], st));
            if (int rc = enqueue_copies(b + 2)) return rc;
        }
        {
            const int v8 = P.nt * 8;
            dim3 grid((3 * v8 * v8 + P.nt * P.nt * 64 + 255) / 256, cnt);
            side_pack_kernel<<<grid, 256, 0, st>>>(d_rj + n0, v, o, P.nt, in.eps_v, in.t1, in.ovov, d_side);
            CU_TRY(cudaGetLastError());
            ++g_launches;
            const int gy = std::max(1, std::min(cnt, kNumSM / P.red_gx));
            reduce_kernel<TS><<<dim3(P.red_gx, gy), RED_THREADS, RedCfg<TS>::SMEM_BYTES, st>>>(
                d_rj + n0, cnt, d_orb, P.norb, v, P.nt, in.eps_o, d_side, d_part);
            CU_TRY(cudaGetLastError());
            ++g_launches;
        }
        if (prof) CU_TRY(cudaEventRecord(e[2], st));
        finalize_kernel<<<cnt, 128, 0, st>>>(d_fj + n0, d_part, P.red_gx * kRedWarps, e_trip);
        CU_TRY(cudaGetLastError());
        ++g_launches;
        if (prof) {
            CU_TRY(cudaEventRecord(e[3], st));
            for (int x = 0; x < 5; ++x) evs.push_back(e[x]);
        }
    }
    if (streamed) {   // later work on `st` (the caller's, or the next call) starts after the copy stream has drained
        cudaEvent_t ev_end;
        if (int rc = event_pool().get(&ev_end)) return rc;
        CU_TRY(cudaEventRecord(ev_end, cs));
        CU_TRY(cudaStreamWaitEvent(st, ev_end, 0));
    }
    if (prof) {
        CU_TRY(cudaStreamSynchronize(st));
        double t_gemm = 0, t_red = 0, t_fin = 0, t_slices = 0;
        float ms = 0;
        for (size_t b = 0; b < nbatch; ++b) {
            CU_TRY(cudaEventElapsedTime(&ms, evs[5 * b + 4], evs[5 * b + 0])); t_slices += ms;
            CU_TRY(cudaEventElapsedTime(&ms, evs[5 * b + 0], evs[5 * b + 1])); t_gemm += ms;
            CU_TRY(cudaEventElapsedTime(&ms, evs[5 * b + 1], evs[5 * b + 2])); t_red += ms;
            CU_TRY(cudaEventElapsedTime(&ms, evs[5 * b + 2], evs[5 * b + 3])); t_fin += ms;
        }
        CU_TRY(cudaEventElapsedTime(&ms, ev_p0, ev_p1));
        const double v3 = (double)v * v * v;
        std::memset(g_prof, 0, sizeof g_prof);
        g_prof[0] = ms;
        g_prof[1] = t_gemm; g_prof[2] = (double)nbatch;
        g_prof[3] = t_red;  g_prof[4] = (double)nbatch;
        g_prof[5] = t_fin;  g_prof[6] = (double)nbatch;
        g_prof[7] = (double)gj.size() * 4.0 * v3 * ((double)v + o);
        g_prof[8] = distinct_u * v3 * sizeof(TS) + (double)nwork * (3.0 * v * v + 4.0 * v) * 8.0;
        g_prof[9] = (double)nwork;
        g_prof[10] = t_slices;
        g_prof[11] = (double)B.loads.size();
        g_prof[12] = h2d_bytes;
        g_prof[13] = ri ? (double)B.loads.size() * 2.0 * P.naux * v3 : 0.0;
        g_prof_valid = true;
    }
    return TRIPLES_OK;
}

int validate_common(int o, int v, int prec, const void* const* ptrs, int nptr, const void* ws, Plan& P,
                    int mode = SLICES_RESIDENT, int nslots = 0, int naux = 0, int win_cap = 0) {
    if (!make_plan(o, v, prec, P, mode, nslots, naux, win_cap))
        return fail(TRIPLES_EINVAL, "invalid sizes/precision: nocc=%d nvirt=%d precision=%d naux=%d (need 1<=nocc<=%d, 1<=nvirt<=%d)",
                    o, v, prec, naux, kMaxOcc, kMaxVirt);
    for (int n = 0; n < nptr; ++n)
        if (!ptrs[n]) return fail(TRIPLES_EINVAL, "null pointer argument (#%d)", n);
    if (!ws) return fail(TRIPLES_EINVAL, "null workspace");
    if (reinterpret_cast<uintptr_t>(ws) & 255) return fail(TRIPLES_EINVAL, "workspace must be 256-byte aligned");
    return TRIPLES_OK;
}

// device-pointer arguments: 16-byte aligned memory of the current device
int check_device_inputs(const void* const* ptrs, int nptr, const void* ws) {
    for (int n = 0; n < nptr; ++n) {
        if (misaligned(ptrs[n])) return fail(TRIPLES_EINVAL, "input pointer #%d is not 16-byte aligned", n);
        if (int rc = check_device_ptr(ptrs[n], "input pointer", n)) return rc;
    }
    return check_device_ptr(ws, "workspace", 0);
}

int dispatch_batches(const Plan& P, const Inputs& in, const Source& src, uint8_t* ws, cudaStream_t st,
                     const std::vector<Triplet>& trip, double* e_trip, size_t rows, const RunOpts& opt = RunOpts()) {
    const int rc = P.prec != TRIPLES_MIXED ? run_batches<double>(P, in, src, ws, st, trip, e_trip, rows, opt)
                                           : run_batches<float>(P, in, src, ws, st, trip, e_trip, rows, opt);
    if (rc != TRIPLES_OK && P.mode == SLICES_STREAMED) {
        // an error in the middle of a streamed run may leave slice copies queued on the library's copy stream: they
        // must not keep writing into the caller's workspace after this call has returned
        const std::string msg = g_err;
        cudaStream_t cs = nullptr;
        if (copy_stream(&cs) == TRIPLES_OK) cudaStreamSynchronize(cs);
        cudaStreamSynchronize(st);
        cudaGetLastError();
        g_err = msg;
    }
    return rc;
}

// all restricted triplets -> e_trip rows, total, results to the caller
int run_full(const Plan& P, const Inputs& in, const Source& src, uint8_t* ws, cudaStream_t st, const RunOpts& opt,
             double* e_out, double* e_triplet_out) {
    std::vector<Triplet> trip;
    enumerate_triplets(P.o, trip);
    double* e_trip = reinterpret_cast<double*>(ws + P.off_etrip);
    double* d_res = reinterpret_cast<double*>(ws + P.off_result);
    g_prof_valid = false;
    g_launches = 0;
    if (int rc = dispatch_batches(P, in, src, ws, st, trip, e_trip, (size_t)P.T, opt)) return rc;
    total_kernel<<<1, 256, 0, st>>>(e_trip, P.T, d_res);
    CU_TRY(cudaGetLastError());
    ++g_launches;
    if (e_triplet_out)
        CU_TRY(cudaMemcpyAsync(e_triplet_out, e_trip, (size_t)P.T * 3 * sizeof(double), cudaMemcpyDeviceToDevice, st));
    CU_TRY(cudaMemcpyAsync(e_out, d_res, 3 * sizeof(double), cudaMemcpyDeviceToHost, st));
    // a caller-supplied maximum of the streamed tensor fixes the operand scale of the packed paths unchecked: an
    // element beyond it overflows FP16 (mixed) or wraps the top digit (emulated FP64) -- pack_xk_kernel flags it
    unsigned int overflow = 0;
    const bool trusted_max = src.mode == SLICES_STREAMED && src.absmax > 0.0 && P.prec != TRIPLES_FP64;
    if (trusted_max)
        CU_TRY(cudaMemcpyAsync(&overflow, reinterpret_cast<const unsigned int*>(ws + P.off_result + 64) + kOverflowWord,
                               sizeof overflow, cudaMemcpyDeviceToHost, st));
    CU_TRY(cudaStreamSynchronize(st));
    if (overflow)
        return fail(TRIPLES_EINVAL, "vvvo_absmax = %g is smaller than the largest |(ab|ck)| of vovv_host: the packed operands "
                    "overflowed and the energies are invalid (pass the true maximum, or <= 0 to let the library scan)",
                    src.absmax);
    return TRIPLES_OK;
}

// The streamed / RI plan for a workspace of `bytes`: the widest window whose minimum cache fits, then as many cache
// slots as fit.  Returns false if not even window 1 fits.
bool fit_plan(int o, int v, int prec, int mode, int naux, size_t bytes, Plan& P) {
    for (int win = 4; win >= 1; --win) {
        Plan M;
        if (!make_plan(o, v, prec, M, mode, 0, naux, win)) return false;
        if (M.win < win) continue;                 // capped already (U budget or o): same plan as a smaller cap
        if (M.total > bytes) continue;
        // X and XT slot of one slice in operand words (osz: 8 FP64, 4 on both packed paths), before alignment: the
        // start of a walk down, so it must not be an under-estimate of the slots that fit
        const size_t per_slot = 2 * M.n_slice * M.osz;
        long long n = M.nslots + (long long)((bytes - M.total) / per_slot) + 1;
        if (n > o) n = o;
        for (; n >= M.nslots; --n)
            if (make_plan(o, v, prec, P, mode, (int)n, naux, win) && P.total <= bytes) return true;
    }
    return false;
}

// Device address of g_noalloc_scratch on the current device: looked up once per device (with that device current),
// then served from the table.  cudaGetSymbolAddress may load the module, hence "first call outside stream capture".
int noalloc_scratch(uint8_t** out) {
    static std::mutex mu;
    static std::map<int, uint8_t*> addr;
    int dev = 0;
    CU_TRY(cudaGetDevice(&dev));
    std::lock_guard<std::mutex> lk(mu);
    auto it = addr.find(dev);
    if (it == addr.end()) {
        void* p = nullptr;
        CU_TRY(cudaGetSymbolAddress(&p, g_noalloc_scratch));
        if (!p || (reinterpret_cast<uintptr_t>(p) & 255))
            return fail(TRIPLES_ECUDA, "cudaGetSymbolAddress gave %p for the static scratch array on device %d", p, dev);
        it = addr.emplace(dev, static_cast<uint8_t*>(p)).first;
    }
    *out = it->second;
    return TRIPLES_OK;
}

template <int KIND>
int run_tc_probe(int clusters, int batches, unsigned long long* out, cudaStream_t st) {
    cudaLaunchConfig_t cfg = {};
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = 2; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.blockDim = dim3(TCP_THREADS);
    cfg.gridDim = dim3((unsigned)clusters * 2);
    cfg.dynamicSmemBytes = 0;
    cfg.stream = st;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    CU_TRY(cudaLaunchKernelEx(&cfg, tc_peak_kernel<KIND>, batches, out));
    ++g_launches;
    return TRIPLES_OK;
}

}  // namespace

// =============================================================================================== C ABI
extern "C" {

int triples_abi_version(void) { return 2; }

long long triples_last_launch_count(void) { return g_launches; }

const char* triples_last_error(void) { return g_err.c_str(); }

void triples_set_profiling(int on) { g_profiling = on; }

int triples_last_profile(double* out16) {
    if (!out16 || !g_prof_valid) return fail(TRIPLES_EINVAL, "no profiled call on this thread");
    std::memcpy(out16, g_prof, sizeof g_prof);
    return TRIPLES_OK;
}

long long triples_triplet_count(int nocc) { return tb::triplet_count(nocc); }

int triples_triplet_list(int nocc, int* ijk_out) {
    if (nocc < 1 || !ijk_out) return fail(TRIPLES_EINVAL, "triples_triplet_list: bad arguments");
    std::vector<Triplet> t;
    enumerate_triplets(nocc, t);
    for (size_t n = 0; n < t.size(); ++n) { ijk_out[3 * n] = t[n].i; ijk_out[3 * n + 1] = t[n].j; ijk_out[3 * n + 2] = t[n].k; }
    return TRIPLES_OK;
}

long long triples_plan_batches(int nocc, int nvirt, int precision, int* batch_of_triplet, int* jobs_out,
                               long long* njobs_out) {
    Plan P;
    if (!make_plan(nocc, nvirt, precision, P)) {
        fail(TRIPLES_EINVAL, "invalid sizes/precision: nocc=%d nvirt=%d precision=%d", nocc, nvirt, precision);
        return -1;
    }
    std::vector<Triplet> trip;
    enumerate_triplets(nocc, trip);
    BatchPlan B;
    build_batches(P, trip, B);
    const size_t nbatch = B.bstart.size() - 1;
    if (batch_of_triplet) {
        for (long long n = 0; n < P.T; ++n) batch_of_triplet[n] = -1;
        for (size_t b = 0; b < nbatch; ++b)
            for (size_t n = B.bstart[b]; n < B.bstart[b + 1]; ++n) batch_of_triplet[B.work[n].index] = (int)b;
    }
    if (jobs_out)
        for (size_t b = 0; b < nbatch; ++b)
            for (int g = B.jstart[b]; g < B.jstart[b + 1]; ++g) {
                const JobDesc& d = B.jobs[g];
                int* o6 = jobs_out + 6 * (size_t)g;
                o6[0] = (int)b; o6[1] = d.p; o6[2] = d.q; o6[3] = d.r; o6[4] = d.gstart; o6[5] = d.gsize;
            }
    if (njobs_out) *njobs_out = (long long)B.jobs.size();
    return (long long)nbatch;
}

long long triples_plan_shards(int nocc, int nvirt, int precision, int nshards, int* shard_of_triplet,
                              long long* jobs_per_shard) {
    Plan P;
    if (!make_plan(nocc, nvirt, precision, P) || nshards < 1) {
        fail(TRIPLES_EINVAL, "invalid sizes/precision/shards: nocc=%d nvirt=%d precision=%d nshards=%d", nocc, nvirt,
             precision, nshards);
        return -1;
    }
    std::vector<Triplet> trip;
    enumerate_triplets(nocc, trip);
    BatchPlan B;
    build_batches(P, trip, B);
    if (shard_of_triplet)
        for (long long n = 0; n < P.T; ++n) shard_of_triplet[n] = -1;
    for (int s = 0; s < nshards; ++s) {
        size_t b0, b1;
        shard_range(B, s, nshards, b0, b1);
        if (shard_of_triplet)
            for (size_t b = b0; b < b1; ++b)
                for (size_t n = B.bstart[b]; n < B.bstart[b + 1]; ++n) shard_of_triplet[B.work[n].index] = s;
        if (jobs_per_shard) jobs_per_shard[s] = (long long)B.jstart[b1] - B.jstart[b0];
    }
    return (long long)(B.bstart.size() - 1);
}

long long triples_plan_slices(int nocc, int nvirt, int precision, int mode, int nslots, int win, int* loads_out,
                              long long loads_cap, int* jobs_out, long long jobs_cap, int* nslots_out) {
    Plan P;
    if (mode != SLICES_STREAMED && mode != SLICES_RI) { fail(TRIPLES_EINVAL, "mode must be 1 (streamed) or 2 (RI)"); return -1; }
    if (!make_plan(nocc, nvirt, precision, P, mode, nslots, mode == SLICES_RI ? 1 : 0, win)) {
        fail(TRIPLES_EINVAL, "invalid sizes/precision: nocc=%d nvirt=%d precision=%d", nocc, nvirt, precision);
        return -1;
    }
    std::vector<Triplet> trip;
    enumerate_triplets(nocc, trip);
    BatchPlan B;
    build_batches(P, trip, B);
    if (!build_slices(nocc, P.nslots, mode == SLICES_STREAMED, B)) { fail(TRIPLES_EWORKSPACE, "slice cache too small"); return -1; }
    const size_t nbatch = B.bstart.size() - 1;
    if (loads_out)
        for (size_t b = 0; b < nbatch; ++b)
            for (int l = B.lstart[b]; l < B.lstart[b + 1] && l < loads_cap; ++l) {
                loads_out[3 * (size_t)l] = (int)b; loads_out[3 * (size_t)l + 1] = B.loads[l].r;
                loads_out[3 * (size_t)l + 2] = B.loads[l].slot;
            }
    if (jobs_out)
        for (size_t b = 0; b < nbatch; ++b)
            for (int g = B.jstart[b]; g < B.jstart[b + 1] && g < jobs_cap; ++g) {
                int* o5 = jobs_out + 5 * (size_t)g;
                o5[0] = (int)b; o5[1] = B.jobs[g].q; o5[2] = B.jobs[g].r; o5[3] = B.jobs[g].xq; o5[4] = B.jobs[g].xr;
            }
    if (nslots_out) { nslots_out[0] = P.nslots; nslots_out[1] = P.win; nslots_out[2] = (int)nbatch; nslots_out[3] = (int)B.jobs.size(); }
    return (long long)B.loads.size();
}

size_t triples_workspace_bytes(int nocc, int nvirt, int precision) {
    Plan P;
    return make_plan(nocc, nvirt, precision, P) ? P.total : 0;
}

size_t triples_workspace_bytes_host(int nocc, int nvirt, int precision) {
    Plan P;
    return make_plan(nocc, nvirt, precision, P) ? P.total_host : 0;
}

size_t triples_workspace_bytes_streamed(int nocc, int nvirt, int precision, int nslots, int win) {
    Plan P;
    return make_plan(nocc, nvirt, precision, P, SLICES_STREAMED, nslots < 0 ? 0 : nslots, 0, win) ? P.total : 0;
}

size_t triples_workspace_bytes_ri(int nocc, int nvirt, int naux, int precision, int nslots, int win) {
    Plan P;
    return make_plan(nocc, nvirt, precision, P, SLICES_RI, nslots < 0 ? 0 : nslots, naux, win) ? P.total : 0;
}

int triples_cache_slots(int nocc, int nvirt, int naux, int precision, int mode, size_t workspace_bytes, int* win_out) {
    if (mode != SLICES_STREAMED && mode != SLICES_RI) return 0;
    Plan P;
    if (!fit_plan(nocc, nvirt, precision, mode, naux, workspace_bytes, P)) return 0;
    if (win_out) *win_out = P.win;
    return P.nslots;
}

int triples_energy_sharded(int nocc, int nvirt, const double* eps_o, const double* eps_v, const double* t1,
                           const double* t2, const double* vvvo, const double* ovoo, const double* ovov, int precision,
                           int shard, int nshards, void* workspace, size_t workspace_bytes, void* cuda_stream,
                           double* e_out, double* e_triplet_out) {
    Plan P;
    const void* ptrs[8] = {eps_o, eps_v, t1, t2, vvvo, ovoo, ovov, e_out};
    if (int rc = validate_common(nocc, nvirt, precision, ptrs, 8, workspace, P)) return rc;
    if (nshards < 1 || shard < 0 || shard >= nshards) return fail(TRIPLES_EINVAL, "shard %d of %d", shard, nshards);
    if (workspace_bytes < P.total)
        return fail(TRIPLES_EWORKSPACE, "workspace too small: %zu bytes given, %zu needed", workspace_bytes, P.total);
    if (int rc = check_device()) return rc;
    if (int rc = check_device_inputs(ptrs, 7, workspace)) return rc;
    if (e_triplet_out)
        if (int rc = check_device_ptr(e_triplet_out, "e_triplet_out", 0)) return rc;
    Inputs in{eps_o, eps_v, t1, t2, ovoo, ovov};
    Source src;
    src.vvvo = vvvo;
    RunOpts opt{shard, nshards};
    return run_full(P, in, src, static_cast<uint8_t*>(workspace), static_cast<cudaStream_t>(cuda_stream), opt, e_out,
                    e_triplet_out);
}

int triples_energy(int nocc, int nvirt, const double* eps_o, const double* eps_v, const double* t1, const double* t2,
                   const double* vvvo, const double* ovoo, const double* ovov, int precision, void* workspace,
                   size_t workspace_bytes, void* cuda_stream, double* e_out, double* e_triplet_out) {
    return triples_energy_sharded(nocc, nvirt, eps_o, eps_v, t1, t2, vvvo, ovoo, ovov, precision, 0, 1, workspace,
                                  workspace_bytes, cuda_stream, e_out, e_triplet_out);
}

// triples_energy on the library's own static scratch array (header: who needs this, the 32 MiB limit, first-call
// set-up, sharing).  Nothing on this path allocates: no cudaMalloc / cudaFree, no stream or event creation.
int triples_energy_noalloc(int nocc, int nvirt, const double* eps_o, const double* eps_v, const double* t1,
                           const double* t2, const double* vvvo, const double* ovoo, const double* ovov, int precision,
                           void* cuda_stream, double* e_out, double* e_triplet_out) {
    // the widest window block whose workspace fits the array (a narrower window = fewer U buffers in flight)
    Plan P, M;
    bool valid = false, fits = false;
    for (int win = 4; win >= 1 && !fits; --win) {
        if (!make_plan(nocc, nvirt, precision, M, SLICES_RESIDENT, 0, 0, win)) break;
        valid = true;
        if (M.win == win && M.total <= (size_t)TRIPLES_NOALLOC_SCRATCH_BYTES) { P = M; fits = true; }
    }
    if (!valid)
        return fail(TRIPLES_EINVAL, "invalid sizes/precision: nocc=%d nvirt=%d precision=%d (need 1<=nocc<=%d, 1<=nvirt<=%d)",
                    nocc, nvirt, precision, kMaxOcc, kMaxVirt);
    if (!fits)    // M is the window-1 plan here: the least this problem can do with
        return fail(TRIPLES_EWORKSPACE,
                    "nocc=%d nvirt=%d precision=%d needs %zu bytes of scratch; the static array of triples_energy_noalloc "
                    "holds %zu: use triples_energy with a workspace", nocc, nvirt, precision, M.total,
                    (size_t)TRIPLES_NOALLOC_SCRATCH_BYTES);
    const void* ptrs[8] = {eps_o, eps_v, t1, t2, vvvo, ovoo, ovov, e_out};
    for (int n = 0; n < 8; ++n)
        if (!ptrs[n]) return fail(TRIPLES_EINVAL, "null pointer argument (#%d)", n);
    if (int rc = check_device()) return rc;
    for (int n = 0; n < 7; ++n) {
        if (misaligned(ptrs[n])) return fail(TRIPLES_EINVAL, "input pointer #%d is not 16-byte aligned", n);
        if (int rc = check_device_ptr(ptrs[n], "input pointer", n)) return rc;
    }
    if (e_triplet_out)
        if (int rc = check_device_ptr(e_triplet_out, "e_triplet_out", 0)) return rc;
    uint8_t* ws = nullptr;
    if (int rc = noalloc_scratch(&ws)) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    // the array still holds the previous call's operands, U buffers and tables (possibly of another shape or
    // precision): everything this run is going to touch starts from zero
    CU_TRY(cudaMemsetAsync(ws, 0, P.total, st));
    Inputs in{eps_o, eps_v, t1, t2, ovoo, ovov};
    Source src;
    src.vvvo = vvvo;
    const int profiling = g_profiling;     // profiling takes events from a pool that grows with cudaEventCreate
    g_profiling = 0;
    const int rc = run_full(P, in, src, ws, st, RunOpts(), e_out, e_triplet_out);
    g_profiling = profiling;
    return rc;
}

int triples_energy_host(int nocc, int nvirt, const double* eps_o, const double* eps_v, const double* t1,
                        const double* t2, const double* vvvo, const double* ovoo, const double* ovov, int precision,
                        void* workspace, size_t workspace_bytes, void* cuda_stream, double* e_out,
                        double* e_triplet_out) {
    Plan P;
    const void* ptrs[8] = {eps_o, eps_v, t1, t2, vvvo, ovoo, ovov, e_out};
    if (int rc = validate_common(nocc, nvirt, precision, ptrs, 8, workspace, P)) return rc;
    if (workspace_bytes < P.total_host)
        return fail(TRIPLES_EWORKSPACE, "workspace too small: %zu bytes given, %zu needed", workspace_bytes, P.total_host);
    if (int rc = check_device()) return rc;
    if (int rc = check_device_ptr(workspace, "workspace", 0)) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    uint8_t* ws = static_cast<uint8_t*>(workspace);
    const double* dev[7];
    for (int n = 0; n < 7; ++n) {
        CU_TRY(cudaMemcpyAsync(ws + P.off_in[n], ptrs[n], P.in_bytes[n], cudaMemcpyHostToDevice, st));
        dev[n] = reinterpret_cast<const double*>(ws + P.off_in[n]);
    }
    int rc = triples_energy(nocc, nvirt, dev[0], dev[1], dev[2], dev[3], dev[4], dev[5], dev[6], precision, workspace,
                            P.total, cuda_stream, e_out, nullptr);
    if (rc) return rc;
    if (e_triplet_out) {
        CU_TRY(cudaMemcpyAsync(e_triplet_out, ws + P.off_etrip, (size_t)P.T * 3 * sizeof(double), cudaMemcpyDeviceToHost, st));
        CU_TRY(cudaStreamSynchronize(st));
    }
    return TRIPLES_OK;
}

int triples_energy_streamed(int nocc, int nvirt, const double* eps_o, const double* eps_v, const double* t1,
                            const double* t2, const double* vovv_host, const double* ovoo, const double* ovov,
                            int precision, double vvvo_absmax, void* workspace, size_t workspace_bytes,
                            void* cuda_stream, double* e_out, double* e_triplet_out) {
    const void* ptrs[8] = {eps_o, eps_v, t1, t2, ovoo, ovov, vovv_host, e_out};
    Plan P0, P;
    if (int rc = validate_common(nocc, nvirt, precision, ptrs, 8, workspace, P0, SLICES_STREAMED, 0, 0, 1)) return rc;
    if (!fit_plan(nocc, nvirt, precision, SLICES_STREAMED, 0, workspace_bytes, P))
        return fail(TRIPLES_EWORKSPACE, "workspace too small: %zu bytes given, %zu needed for window 1 with %d cache slots",
                    workspace_bytes, P0.total, P0.nslots);
    if (int rc = check_device()) return rc;
    if (int rc = check_device_inputs(ptrs, 6, workspace)) return rc;
    if (e_triplet_out)
        if (int rc = check_device_ptr(e_triplet_out, "e_triplet_out", 0)) return rc;
    Inputs in{eps_o, eps_v, t1, t2, ovoo, ovov};
    Source src;
    src.mode = SLICES_STREAMED;
    src.vovv_host = vovv_host;
    src.absmax = vvvo_absmax;
    return run_full(P, in, src, static_cast<uint8_t*>(workspace), static_cast<cudaStream_t>(cuda_stream), RunOpts(),
                    e_out, e_triplet_out);
}

int triples_energy_ri(int nocc, int nvirt, int naux, const double* eps_o, const double* eps_v, const double* t1,
                      const double* t2, const double* B, const double* ovoo, const double* ovov, int precision,
                      void* workspace, size_t workspace_bytes, void* cuda_stream, double* e_out,
                      double* e_triplet_out) {
    const void* ptrs[8] = {eps_o, eps_v, t1, t2, B, ovoo, ovov, e_out};
    Plan P0, P;
    if (int rc = validate_common(nocc, nvirt, precision, ptrs, 8, workspace, P0, SLICES_RI, 0, naux, 1)) return rc;
    if (!fit_plan(nocc, nvirt, precision, SLICES_RI, naux, workspace_bytes, P))
        return fail(TRIPLES_EWORKSPACE, "workspace too small: %zu bytes given, %zu needed for window 1 with %d cache slots",
                    workspace_bytes, P0.total, P0.nslots);
    if (int rc = check_device()) return rc;
    if (int rc = check_device_inputs(ptrs, 7, workspace)) return rc;
    if (e_triplet_out)
        if (int rc = check_device_ptr(e_triplet_out, "e_triplet_out", 0)) return rc;
    Inputs in{eps_o, eps_v, t1, t2, ovoo, ovov};
    Source src;
    src.mode = SLICES_RI;
    src.B = B;
    return run_full(P, in, src, static_cast<uint8_t*>(workspace), static_cast<cudaStream_t>(cuda_stream), RunOpts(),
                    e_out, e_triplet_out);
}

int triples_energy_subset(int nocc, int nvirt, const double* eps_o, const double* eps_v, const double* t1,
                          const double* t2, const double* vvvo, const double* ovoo, const double* ovov, int precision,
                          int ntrip, const int* ijk, void* workspace, size_t workspace_bytes, void* cuda_stream,
                          double* e_out) {
    Plan P;
    const void* ptrs[7] = {eps_o, eps_v, t1, t2, vvvo, ovoo, ovov};
    if (int rc = validate_common(nocc, nvirt, precision, ptrs, 7, workspace, P)) return rc;
    if (ntrip < 0 || (ntrip > 0 && (!ijk || !e_out))) return fail(TRIPLES_EINVAL, "bad triplet list");
    if ((long long)ntrip > P.T) return fail(TRIPLES_EINVAL, "more triplets (%d) than the restricted loop has (%lld)", ntrip, P.T);
    if (workspace_bytes < P.total)
        return fail(TRIPLES_EWORKSPACE, "workspace too small: %zu bytes given, %zu needed", workspace_bytes, P.total);
    std::vector<Triplet> trip(ntrip);
    for (int n = 0; n < ntrip; ++n) {
        const int i = ijk[3 * n], j = ijk[3 * n + 1], k = ijk[3 * n + 2];
        if (i < 0 || i > j || j > k || k >= nocc) return fail(TRIPLES_EINVAL, "triplet #%d = (%d,%d,%d) is not 0<=i<=j<=k<nocc", n, i, j, k);
        trip[n] = {i, j, k, n};
    }
    if (ntrip == 0) return TRIPLES_OK;
    if (int rc = check_device()) return rc;
    if (int rc = check_device_inputs(ptrs, 7, workspace)) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    uint8_t* ws = static_cast<uint8_t*>(workspace);
    double* e_trip = reinterpret_cast<double*>(ws + P.off_etrip);
    Inputs in{eps_o, eps_v, t1, t2, ovoo, ovov};
    Source src;
    src.vvvo = vvvo;
    g_prof_valid = false;
    g_launches = 0;
    if (int rc = dispatch_batches(P, in, src, ws, st, trip, e_trip, (size_t)ntrip)) return rc;
    CU_TRY(cudaMemcpyAsync(e_out, e_trip, (size_t)ntrip * 3 * sizeof(double), cudaMemcpyDeviceToHost, st));
    CU_TRY(cudaStreamSynchronize(st));
    return TRIPLES_OK;
}

int triples_w_block(int nocc, int nvirt, const double* t2, const double* vvvo, const double* ovoo, int precision,
                    int i, int j, int k, void* workspace, size_t workspace_bytes, void* cuda_stream, double* W_out) {
    Plan P;
    const void* ptrs[4] = {t2, vvvo, ovoo, W_out};
    if (int rc = validate_common(nocc, nvirt, precision, ptrs, 4, workspace, P)) return rc;
    if (i < 0 || j < 0 || k < 0 || i >= nocc || j >= nocc || k >= nocc) return fail(TRIPLES_EINVAL, "occupied index out of range");
    if (workspace_bytes < P.total)
        return fail(TRIPLES_EWORKSPACE, "workspace too small: %zu bytes given, %zu needed", workspace_bytes, P.total);
    if (int rc = check_device()) return rc;
    if (int rc = check_device_inputs(ptrs, 4, workspace)) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    uint8_t* ws = static_cast<uint8_t*>(workspace);
    Operands op = carve_operands(P, ws);
    g_launches = 0;
    event_pool().reset();
    Inputs in{nullptr, nullptr, nullptr, t2, ovoo, nullptr};
    Source src;
    src.vvvo = vvvo;
    if (int rc = run_prepare(P, in, src, op, st, nullptr)) return rc;
    Maps maps;
    if (int rc = build_maps(P, op, &maps)) return rc;
    uint8_t* ubase = ws + P.off_u;
    const size_t ub = (size_t)UBLK * P.esz;   // U1, U2, U3 blocks of a tile are adjacent
    GemmJob gj[3] = {{i, j, k, 0, ubase, nullptr, 1, k, j, 0},          // three groups of one job
                     {j, i, k, 1, ubase + ub, nullptr, 1, k, i, 0},
                     {k, i, j, 2, ubase + 2 * ub, nullptr, 1, j, i, 0}};
    GemmJob* d_gj = reinterpret_cast<GemmJob*>(ws + P.off_gjobs);
    CU_TRY(cudaMemcpyAsync(d_gj, gj, sizeof gj, cudaMemcpyHostToDevice, st));
    if (int rc = launch_gemm(P, maps, op, d_gj, 3, st)) return rc;
    if (P.esz == 8)
        assemble_w_kernel<double><<<kNumSM * 4, 256, 0, st>>>((const double*)ubase, nvirt, P.nt, W_out);
    else
        assemble_w_kernel<float><<<kNumSM * 4, 256, 0, st>>>((const float*)ubase, nvirt, P.nt, W_out);
    CU_TRY(cudaGetLastError());
    ++g_launches;
    CU_TRY(cudaStreamSynchronize(st));
    return TRIPLES_OK;
}

int triples_probe_fp64_peak(void* workspace, size_t workspace_bytes, void* cuda_stream, int iters, double* tflops_out) {
    if (!workspace || !tflops_out || iters < 1) return fail(TRIPLES_EINVAL, "triples_probe_fp64_peak: bad arguments");
    const size_t need = (size_t)kNumSM * PROBE_THREADS * sizeof(double);
    if (workspace_bytes < need) return fail(TRIPLES_EWORKSPACE, "workspace too small: %zu bytes given, %zu needed", workspace_bytes, need);
    if (int rc = check_device()) return rc;
    if (int rc = check_device_ptr(workspace, "workspace", 0)) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    event_pool().reset();
    cudaEvent_t e0, e1;
    if (int rc = event_pool().get(&e0)) return rc;
    if (int rc = event_pool().get(&e1)) return rc;
    double best = 0.0;
    for (int rep = 0; rep < 4; ++rep) {      // the first repetition warms the clocks up
        CU_TRY(cudaEventRecord(e0, st));
        fp64_peak_kernel<<<kNumSM, PROBE_THREADS, 0, st>>>(static_cast<double*>(workspace), iters);
        CU_TRY(cudaGetLastError());
        CU_TRY(cudaEventRecord(e1, st));
        CU_TRY(cudaStreamSynchronize(st));
        float ms = 0;
        CU_TRY(cudaEventElapsedTime(&ms, e0, e1));
        // m8n8k4: 512 flop per warp instruction = 16 per thread
        const double tf = (double)kNumSM * PROBE_THREADS * (double)iters * PROBE_ACC * 16.0 / (ms * 1e-3) / 1e12;
        if (rep > 0 && tf > best) best = tf;
    }
    g_launches = 4;
    *tflops_out = best;
    return TRIPLES_OK;
}

int triples_probe_tc_peak(int kind, double seconds, void* workspace, size_t workspace_bytes, void* cuda_stream,
                          double* tops_out, double* sm_mhz_out) {
    if (!workspace || !tops_out || (kind != 0 && kind != 1) || !(seconds > 0.0) || seconds > 10.0)
        return fail(TRIPLES_EINVAL, "triples_probe_tc_peak: bad arguments (kind 0 | 1, 0 < seconds <= 10)");
    const size_t need = (size_t)kNumSM * sizeof(unsigned long long);
    if (workspace_bytes < need) return fail(TRIPLES_EWORKSPACE, "workspace too small: %zu bytes given, %zu needed", workspace_bytes, need);
    if (int rc = check_device()) return rc;
    if (int rc = check_device_ptr(workspace, "workspace", 0)) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    unsigned long long* out = static_cast<unsigned long long*>(workspace);
    // as many CTA pairs as are co-resident (what the contraction kernels get too)
    int clusters = 0;
    {
        cudaLaunchConfig_t cfg = {};
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = 2; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
        cfg.blockDim = dim3(TCP_THREADS);
        cfg.attrs = attr;
        cfg.numAttrs = 1;
        if (kind == 0) { if (int rc = max_pair_clusters(tc_peak_kernel<0>, 6, cfg, 2, &clusters)) return rc; }
        else { if (int rc = max_pair_clusters(tc_peak_kernel<1>, 7, cfg, 2, &clusters)) return rc; }
    }
    event_pool().reset();
    cudaEvent_t e0, e1;
    if (int rc = event_pool().get(&e0)) return rc;
    if (int rc = event_pool().get(&e1)) return rc;
    g_launches = 0;
    const double ops_per_batch = (double)clusters * TCP_BATCH * 2.0 * 256.0 * (kind == 0 ? 256.0 * 16.0 : 80.0 * 32.0);
    int batches = 2000;                       // calibration run, then one run of about `seconds`
    double tops = 0.0;
    for (int pass = 0; pass < 2; ++pass) {
        CU_TRY(cudaMemsetAsync(out, 0, need, st));
        CU_TRY(cudaEventRecord(e0, st));
        if (int rc = kind == 0 ? run_tc_probe<0>(clusters, batches, out, st) : run_tc_probe<1>(clusters, batches, out, st)) return rc;
        CU_TRY(cudaEventRecord(e1, st));
        CU_TRY(cudaStreamSynchronize(st));
        float ms = 0;
        CU_TRY(cudaEventElapsedTime(&ms, e0, e1));
        tops = ops_per_batch * batches / (ms * 1e-3) / 1e12;
        if (pass == 0) {
            const double want = seconds / (ms * 1e-3) * batches;
            batches = (int)std::min(std::max(want, 2000.0), 1.0e9);
        }
    }
    if (sm_mhz_out) {
        unsigned long long h[2] = {0, 0};
        CU_TRY(cudaMemcpyAsync(h, out, sizeof h, cudaMemcpyDeviceToHost, st));
        CU_TRY(cudaStreamSynchronize(st));
        *sm_mhz_out = h[1] ? (double)h[0] / (double)h[1] * 1e3 : 0.0;
    }
    *tops_out = tops;
    return TRIPLES_OK;
}

}  // extern "C"
