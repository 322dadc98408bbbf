// triples_b200.cu -- C-ABI entry points of include/triples_b200.h and the host-side driver.
// No CPU fallback: every step of the hot path runs in the kernels of gemm_f64.cuh / gemm_tf32.cuh / reduce.cuh.
#include "../../include/triples_b200.h"

#include <cuda.h>
#include <cuda_runtime.h>

#include <algorithm>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <string>
#include <vector>

#include "gemm_f64.cuh"
#include "gemm_tf32.cuh"
#include "plan.h"
#include "prepare.cuh"
#include "reduce.cuh"

namespace {

using namespace tb;

thread_local std::string g_err;
thread_local double g_prof[10];
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
                    CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
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
thread_local EventPool g_events;

// ------------------------------------------------------------------------------------------ contraction launch
template <int WM, int WN, int NT, int STAGES>
int launch_gemm_f64(const GemmMaps& maps, const GemmJob* jobs, int njobs, const Plan& P, cudaStream_t st) {
    using C = GemmF64Cfg<WM, WN, NT, STAGES>;
    auto kern = gemm_f64_kernel<WM, WN, NT, STAGES>;
    static bool attr_set = false;
    if (!attr_set) {
        CU_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM_BYTES));
        attr_set = true;
    }
    const long long items = (long long)P.mtiles * P.ntiles * njobs;
    if (items == 0) return TRIPLES_OK;
    const int grid = (int)std::min<long long>(items, kNumSM);     // persistent: one CTA per SM
    kern<<<grid, C::THREADS, C::SMEM_BYTES, st>>>(maps, jobs, njobs, P.v, P.vp, P.o, P.mtiles, P.ntiles);
    CU_TRY(cudaGetLastError());
    ++g_launches;
    return TRIPLES_OK;
}

struct Operands {   // device pointers of the repacked operands (workspace) for one precision
    void *x, *xt, *ot, *t2;
    void *t2k, *t2kt;   // mixed path only
    float* scales;      // mixed path only: 2^sg, 2^st, 2^-(sg+st) (prepare.cuh scales_kernel), then two uint maxima
};

struct Maps {   // tensor maps of the contraction kernel of the plan's precision
    GemmMaps f64;
    Tf32Maps tf32;
};

int build_maps_f64(const Plan& P, const Operands& op, GemmMaps* maps) {
    const uint64_t o = P.o, v = P.v, vp = P.vp, opp = P.op, N = v * vp;
    const CUtensorMapDataType dt = CU_TENSOR_MAP_DATA_TYPE_FLOAT64;
    int rc;
    if ((rc = make_map3(&maps->t2a, dt, 8, op.t2, v, v, o * o, vp, v * vp, 16, P.BM, 1))) return rc;
    if ((rc = make_map3(&maps->ota, dt, 8, op.ot, o, v, o * o, opp, v * opp, 16, P.BM, 1))) return rc;
    if ((rc = make_map3(&maps->x, dt, 8, op.x, N, v, o, N, v * N, 16, 16, 1))) return rc;
    if ((rc = make_map3(&maps->xt, dt, 8, op.xt, N, v, o, N, v * N, 16, 16, 1))) return rc;
    if ((rc = make_map3(&maps->t2bq, dt, 8, op.t2, N, o, o, N, o * N, 16, 16, 1))) return rc;
    if ((rc = make_map3(&maps->t2br, dt, 8, op.t2, N, o, o, N, o * N, 16, 1, 16))) return rc;
    return TRIPLES_OK;
}

int build_maps_tf32(const Plan& P, const Operands& op, Tf32Maps* maps) {
    const uint64_t o = P.o, v = P.v, vk = P.vk, ok = P.ok, NR = (uint64_t)P.v * P.vp;
    const CUtensorMapDataType dt = CU_TENSOR_MAP_DATA_TYPE_FLOAT32;
    int rc;
    // K extent = v / o: TMA zero-fills the rest of the last 32-wide chunk
    if ((rc = make_map3(&maps->xk, dt, 4, op.x, v, NR, o, vk, NR * vk, TF_BK, TF_BM, 1))) return rc;
    if ((rc = make_map3(&maps->xkt, dt, 4, op.xt, v, NR, o, vk, NR * vk, TF_BK, TF_BM, 1))) return rc;
    if ((rc = make_map3(&maps->t2k, dt, 4, op.t2k, o, NR, o, ok, NR * ok, TF_BK, TF_BM, 1))) return rc;
    if ((rc = make_map3(&maps->t2kt, dt, 4, op.t2kt, o, NR, o, ok, NR * ok, TF_BK, TF_BM, 1))) return rc;
    if ((rc = make_map3(&maps->t2a, dt, 4, op.t2, v, v, o * o, vk, v * vk, TF_BK, P.tf_npad, 1))) return rc;
    if ((rc = make_map3(&maps->ota, dt, 4, op.ot, o, v, o * o, ok, v * ok, TF_BK, P.tf_npad, 1))) return rc;
    return TRIPLES_OK;
}

int build_maps(const Plan& P, const Operands& op, Maps* maps) {
    return P.prec == TRIPLES_FP64 ? build_maps_f64(P, op, &maps->f64) : build_maps_tf32(P, op, &maps->tf32);
}

int launch_gemm_tf32(const Tf32Maps& maps, const GemmJob* jobs, int njobs, const Plan& P, const float* scales,
                     cudaStream_t st) {
    static bool attr_set = false;
    if (!attr_set) {
        CU_TRY(cudaFuncSetAttribute(gemm_tf32_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, TF_SMEM_LIMIT));
        attr_set = true;
    }
    const int cs = P.tf_cs;
    if (njobs > TF_MAX_JOBS) return fail(TRIPLES_EINVAL, "internal: %d contraction jobs in one launch (max %d)", njobs, TF_MAX_JOBS);
    const long long items = (long long)njobs * ((P.tf_mtiles + cs - 1) / cs) * P.tf_ntiles;   // per cluster
    if (items == 0) return TRIPLES_OK;
    cudaLaunchConfig_t cfg = {};
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = cs; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.blockDim = dim3(TF_THREADS);
    cfg.dynamicSmemBytes = tf32_smem_bytes(P.tf_npad);
    cfg.stream = st;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    static int max_clusters = 0;   // co-resident CTA pairs (one CTA per SM)
    if (!max_clusters) {
        cfg.gridDim = dim3(kNumSM / cs * cs);
        int n = 0;
        CU_TRY(cudaOccupancyMaxActiveClusters(&n, gemm_tf32_kernel, &cfg));
        if (n < 1) return fail(TRIPLES_ECUDA, "no CTA pair of the mixed contraction fits the device");
        max_clusters = std::min(n, kNumSM / cs);
    }
    cfg.gridDim = dim3((unsigned)(std::min<long long>(items, max_clusters) * cs));
    CU_TRY(cudaLaunchKernelEx(&cfg, gemm_tf32_kernel, maps, jobs, njobs, P.v, P.vp, P.o, P.tf_mtiles, P.tf_ntiles,
                              P.tf_bn, P.tf_npad, scales));
    ++g_launches;
    return TRIPLES_OK;
}

int launch_gemm(const Plan& P, const Maps& maps, const Operands& op, const GemmJob* jobs, int njobs, cudaStream_t st) {
    if (P.prec == TRIPLES_MIXED) return launch_gemm_tf32(maps.tf32, jobs, njobs, P, op.scales, st);
    switch (P.cfg) {
        case CFG_M120_N128: return launch_gemm_f64<3, 4, 4, 4>(maps.f64, jobs, njobs, P, st);
        case CFG_M80_N192: return launch_gemm_f64<2, 6, 4, 4>(maps.f64, jobs, njobs, P, st);
        default: return launch_gemm_f64<1, 8, 4, 4>(maps.f64, jobs, njobs, P, st);
    }
}

// ------------------------------------------------------------------------------------------ prepare (S0)
// Mixed path: K-major FP32 hi/lo operands of gemm_tf32.cuh.
int run_prepare_mixed(const Plan& P, const double* t2, const double* vvvo, const double* ovoo, const Operands& op,
                      cudaStream_t st) {
    const int o = P.o, v = P.v;
    if (P.vp != v || P.vk != v) {   // pads are zero words (the converter warps treat them as 0)
        CU_TRY(cudaMemsetAsync(op.x, 0, P.n_x * 4, st));
        CU_TRY(cudaMemsetAsync(op.xt, 0, P.n_x * 4, st));
        CU_TRY(cudaMemsetAsync(op.t2, 0, P.n_t2 * 4, st));
    }
    if (P.vp != v || P.ok != o) {
        CU_TRY(cudaMemsetAsync(op.t2k, 0, P.n_t2k * 4, st));
        CU_TRY(cudaMemsetAsync(op.t2kt, 0, P.n_t2k * 4, st));
    }
    if (P.ok != o) CU_TRY(cudaMemsetAsync(op.ot, 0, P.n_ot * 4, st));
    {   // power-of-two scales of the two tensor classes
        unsigned int* mx = reinterpret_cast<unsigned int*>(op.scales + 4);
        CU_TRY(cudaMemsetAsync(mx, 0, 8, st));
        absmax_kernel<<<kNumSM * 8, 256, 0, st>>>(vvvo, (size_t)v * v * v * o, mx);
        absmax_kernel<<<kNumSM, 256, 0, st>>>(ovoo, (size_t)o * v * o * o, mx);
        absmax_kernel<<<kNumSM * 2, 256, 0, st>>>(t2, (size_t)o * o * v * v, mx + 1);
        scales_kernel<<<1, 32, 0, st>>>(mx, op.scales);
        CU_TRY(cudaGetLastError());
        g_launches += 4;
    }
    {
        static bool attr_set = false;
        if (!attr_set) {
            CU_TRY(cudaFuncSetAttribute(pack_xk_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, PKX_SMEM));
            attr_set = true;
        }
        const size_t S = (size_t)v * v * o;
        dim3 grid((unsigned)((S + PKX_SPAN - 1) / PKX_SPAN), (v + 31) / 32);
        pack_xk_kernel<<<grid, 256, PKX_SMEM, st>>>(vvvo, v, P.vp, P.vk, o, (float*)op.x, (float*)op.xt, op.scales);
        CU_TRY(cudaGetLastError());
        ++g_launches;
    }
    {
        dim3 grid(o * v, (v + 63) / 64, (o + 63) / 64);
        pack_t2k_kernel<<<grid, 256, 0, st>>>(t2, v, P.vp, o, P.ok, (float*)op.t2k, (float*)op.t2kt, op.scales + 1);
        CU_TRY(cudaGetLastError());
        ++g_launches;
    }
    pack_ot_kernel<float><<<kNumSM * 4, 256, 0, st>>>(ovoo, v, o, P.ok, (float*)op.ot, op.scales);
    CU_TRY(cudaGetLastError());
    ++g_launches;
    pack_t2_kernel<float><<<kNumSM * 8, 256, 0, st>>>(t2, (size_t)o * o * v, v, P.vk, (float*)op.t2, op.scales + 1);
    CU_TRY(cudaGetLastError());
    ++g_launches;
    return TRIPLES_OK;
}

int run_prepare(const Plan& P, const double* t2, const double* vvvo, const double* ovoo, const Operands& op,
                cudaStream_t st) {
    if (P.prec == TRIPLES_MIXED) return run_prepare_mixed(P, t2, vvvo, ovoo, op, st);
    using TO = double;
    const int o = P.o, v = P.v;
    if (P.vp != v) {   // zero the pad columns (XT: entry c = v of a row is never written by the transpose)
        CU_TRY(cudaMemsetAsync(op.x, 0, P.n_x * sizeof(TO), st));
        CU_TRY(cudaMemsetAsync(op.xt, 0, P.n_x * sizeof(TO), st));
        CU_TRY(cudaMemsetAsync(op.t2, 0, P.n_t2 * sizeof(TO), st));
    }
    if (P.op != o) CU_TRY(cudaMemsetAsync(op.ot, 0, P.n_ot * sizeof(TO), st));
    {   // X
        int RB = 128;
        while ((size_t)RB * (o + 1) * 8 > 64 * 1024 && RB > 1) RB /= 2;
        const size_t R = (size_t)v * v * v;
        const size_t smem = (size_t)RB * (o + 1) * 8;
        auto kern = pack_x_kernel<TO>;
        CU_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024));
        kern<<<(unsigned)((R + RB - 1) / RB), 256, smem, st>>>(vvvo, v, P.vp, o, RB, (TO*)op.x);
        CU_TRY(cudaGetLastError());
        ++g_launches;
    }
    {   // XT
        dim3 grid((v + 31) / 32, (v + 31) / 32, 1);
        for (int r = 0; r < o; ++r) {   // gridDim.z <= 65535: one launch per r-slice
            grid.z = v;
            const size_t sl = (size_t)r * v * v * P.vp;
            transpose_planes_kernel<TO><<<grid, 256, 0, st>>>((const TO*)op.x + sl, v, P.vp, (TO*)op.xt + sl);
            ++g_launches;
        }
        CU_TRY(cudaGetLastError());
    }
    pack_ot_kernel<TO><<<kNumSM * 4, 256, 0, st>>>(ovoo, v, o, P.op, (TO*)op.ot, nullptr);
    CU_TRY(cudaGetLastError());
    ++g_launches;
    pack_t2_kernel<TO><<<kNumSM * 8, 256, 0, st>>>(t2, (size_t)o * o * v, v, P.vp, (TO*)op.t2, nullptr);
    CU_TRY(cudaGetLastError());
    ++g_launches;
    return TRIPLES_OK;
}

Operands carve_operands(const Plan& P, uint8_t* ws) {
    Operands op{};
    op.x = ws + P.off_x; op.xt = ws + P.off_xt; op.ot = ws + P.off_ot; op.t2 = ws + P.off_t2;
    if (P.prec == TRIPLES_MIXED) {
        op.t2k = ws + P.off_t2k; op.t2kt = ws + P.off_t2kt;
        op.scales = reinterpret_cast<float*>(ws + P.off_result + 64);   // the result block has 256 bytes, 24 used
    }
    return op;
}

// ------------------------------------------------------------------------------------------ core driver
struct Inputs {
    const double *eps_o, *eps_v, *t1, *t2, *vvvo, *ovoo, *ovov;
};

// Runs prepare + all batches for `trip` (restricted triplets, index = row of e_trip to write) and leaves the
// weighted per-triplet energies in e_trip (device, 3 doubles per row; rows of i=j=k triplets are zero).
template <typename TS>
int run_batches(const Plan& P, const Inputs& in, uint8_t* ws, cudaStream_t st, const std::vector<Triplet>& trip,
                double* e_trip, size_t e_trip_rows) {
    const int o = P.o, v = P.v;
    Operands op = carve_operands(P, ws);
    const bool prof = g_profiling != 0;
    g_events.reset();
    cudaEvent_t ev_p0 = nullptr, ev_p1 = nullptr;
    if (prof) {
        if (int rc = g_events.get(&ev_p0)) return rc;
        if (int rc = g_events.get(&ev_p1)) return rc;
        CU_TRY(cudaEventRecord(ev_p0, st));
    }
    if (int rc = run_prepare(P, in.t2, in.vvvo, in.ovoo, op, st)) return rc;
    if (prof) CU_TRY(cudaEventRecord(ev_p1, st));

    Maps maps;
    if (int rc = build_maps(P, op, &maps)) return rc;

    // ---- batches and job tables (plan.h), uploaded once
    std::vector<Orbit> orbits;
    enumerate_orbits(v, orbits);
    BatchPlan B;
    build_batches(P, trip, B);
    const std::vector<Triplet>& work = B.work;
    const std::vector<size_t>& bstart = B.bstart;
    const std::vector<int>& gj_begin = B.jstart;
    const size_t nwork = work.size(), nbatch = bstart.size() - 1;
    const double distinct_u = B.distinct_u;
    TS* ubase = reinterpret_cast<TS*>(ws + P.off_u);
    std::vector<GemmJob> gj(B.jobs.size());
    for (size_t n = 0; n < gj.size(); ++n) {
        const JobDesc& d = B.jobs[n];
        TS* ub = ubase + (size_t)3 * d.slot * P.n_u;      // interleaved blocks of U1,U2,U3 of the slot (ulayout.cuh)
        gj[n] = {d.p, d.q, d.r, d.gstart, ub + (size_t)d.u * UBLK, d.u2 < 0 ? nullptr : ub + (size_t)d.u2 * UBLK,
                 d.gsize, {0, 0, 0}};
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
    {
        static bool attr_set = false;
        if (!attr_set) {
            CU_TRY(cudaFuncSetAttribute(reduce_kernel<TS>, cudaFuncAttributeMaxDynamicSharedMemorySize, RedCfg<TS>::SMEM_BYTES));
            attr_set = true;
        }
    }
    FinJob* d_fj = reinterpret_cast<FinJob*>(ws + P.off_fjobs);
    uchar4* d_orb = reinterpret_cast<uchar4*>(ws + P.off_orb);
    double2* d_part = reinterpret_cast<double2*>(ws + P.off_part);
    if (!gj.empty()) CU_TRY(cudaMemcpyAsync(d_gj, gj.data(), gj.size() * sizeof(GemmJob), cudaMemcpyHostToDevice, st));
    if (nwork) {
        CU_TRY(cudaMemcpyAsync(d_rj, rj.data(), nwork * sizeof(RedJob), cudaMemcpyHostToDevice, st));
        CU_TRY(cudaMemcpyAsync(d_fj, fj.data(), nwork * sizeof(FinJob), cudaMemcpyHostToDevice, st));
    }
    CU_TRY(cudaMemcpyAsync(d_orb, orbits.data(), orbits.size() * sizeof(Orbit), cudaMemcpyHostToDevice, st));
    CU_TRY(cudaMemsetAsync(e_trip, 0, e_trip_rows * 3 * sizeof(double), st));

    // ---- batches: contraction -> fused reduction -> per-triplet finalize
    std::vector<cudaEvent_t> evs;
    for (size_t b = 0; b < nbatch; ++b) {
        const size_t n0 = bstart[b];
        const int cnt = (int)(bstart[b + 1] - n0);
        const int g0 = gj_begin[b], g1 = gj_begin[b + 1];
        cudaEvent_t e[4] = {nullptr, nullptr, nullptr, nullptr};
        if (prof) {
            for (int x = 0; x < 4; ++x) if (int rc = g_events.get(&e[x])) return rc;
            CU_TRY(cudaEventRecord(e[0], st));
        }
        if (int rc = launch_gemm(P, maps, op, d_gj + g0, g1 - g0, st)) return rc;
        if (prof) CU_TRY(cudaEventRecord(e[1], st));
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
            for (int x = 0; x < 4; ++x) evs.push_back(e[x]);
        }
    }
    if (prof) {
        CU_TRY(cudaStreamSynchronize(st));
        double t_gemm = 0, t_red = 0, t_fin = 0;
        float ms = 0;
        for (size_t b = 0; b < nbatch; ++b) {
            CU_TRY(cudaEventElapsedTime(&ms, evs[4 * b + 0], evs[4 * b + 1])); t_gemm += ms;
            CU_TRY(cudaEventElapsedTime(&ms, evs[4 * b + 1], evs[4 * b + 2])); t_red += ms;
            CU_TRY(cudaEventElapsedTime(&ms, evs[4 * b + 2], evs[4 * b + 3])); t_fin += ms;
        }
        CU_TRY(cudaEventElapsedTime(&ms, ev_p0, ev_p1));
        const double v3 = (double)v * v * v;
        g_prof[0] = ms;
        g_prof[1] = t_gemm; g_prof[2] = (double)nbatch;
        g_prof[3] = t_red;  g_prof[4] = (double)nbatch;
        g_prof[5] = t_fin;  g_prof[6] = (double)nbatch;
        g_prof[7] = (double)gj.size() * 4.0 * v3 * ((double)v + o);
        g_prof[8] = distinct_u * v3 * sizeof(TS) + (double)nwork * (3.0 * v * v + 4.0 * v) * 8.0;
        g_prof[9] = (double)nwork;
        g_prof_valid = true;
    }
    return TRIPLES_OK;
}

int validate_common(int o, int v, int prec, const void* const* ptrs, int nptr, const void* ws, size_t ws_bytes,
                    size_t need, Plan& P) {
    if (!make_plan(o, v, prec, P))
        return fail(TRIPLES_EINVAL, "invalid sizes/precision: nocc=%d nvirt=%d precision=%d (need 1<=nocc<=%d, 1<=nvirt<=%d)",
                    o, v, prec, kMaxOcc, kMaxVirt);
    for (int n = 0; n < nptr; ++n)
        if (!ptrs[n]) return fail(TRIPLES_EINVAL, "null pointer argument (#%d)", n);
    if (!ws) return fail(TRIPLES_EINVAL, "null workspace");
    if (reinterpret_cast<uintptr_t>(ws) & 255) return fail(TRIPLES_EINVAL, "workspace must be 256-byte aligned");
    (void)need;
    (void)ws_bytes;
    return TRIPLES_OK;
}

int dispatch_batches(const Plan& P, const Inputs& in, uint8_t* ws, cudaStream_t st, const std::vector<Triplet>& trip,
                     double* e_trip, size_t rows) {
    if (P.prec == TRIPLES_FP64) return run_batches<double>(P, in, ws, st, trip, e_trip, rows);
    return run_batches<float>(P, in, ws, st, trip, e_trip, rows);
}

}  // namespace

// =============================================================================================== C ABI
extern "C" {

int triples_abi_version(void) { return 1; }

long long triples_last_launch_count(void) { return g_launches; }

const char* triples_last_error(void) { return g_err.c_str(); }

void triples_set_profiling(int on) { g_profiling = on; }

int triples_last_profile(double* out10) {
    if (!out10 || !g_prof_valid) return fail(TRIPLES_EINVAL, "no profiled call on this thread");
    std::memcpy(out10, g_prof, sizeof g_prof);
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

size_t triples_workspace_bytes(int nocc, int nvirt, int precision) {
    Plan P;
    return make_plan(nocc, nvirt, precision, P) ? P.total : 0;
}

size_t triples_workspace_bytes_host(int nocc, int nvirt, int precision) {
    Plan P;
    return make_plan(nocc, nvirt, precision, P) ? P.total_host : 0;
}

int triples_energy(int nocc, int nvirt, const double* eps_o, const double* eps_v, const double* t1, const double* t2,
                   const double* vvvo, const double* ovoo, const double* ovov, int precision, void* workspace,
                   size_t workspace_bytes, void* cuda_stream, double* e_out, double* e_triplet_out) {
    Plan P;
    const void* ptrs[8] = {eps_o, eps_v, t1, t2, vvvo, ovoo, ovov, e_out};
    if (int rc = validate_common(nocc, nvirt, precision, ptrs, 8, workspace, workspace_bytes, 0, P)) return rc;
    for (int n = 0; n < 7; ++n)
        if (misaligned(ptrs[n])) return fail(TRIPLES_EINVAL, "input pointer #%d is not 16-byte aligned", n);
    if (workspace_bytes < P.total)
        return fail(TRIPLES_EWORKSPACE, "workspace too small: %zu bytes given, %zu needed", workspace_bytes, P.total);
    if (int rc = check_device()) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    uint8_t* ws = static_cast<uint8_t*>(workspace);
    std::vector<Triplet> trip;
    enumerate_triplets(nocc, trip);
    double* e_trip = reinterpret_cast<double*>(ws + P.off_etrip);
    double* d_res = reinterpret_cast<double*>(ws + P.off_result);
    Inputs in{eps_o, eps_v, t1, t2, vvvo, ovoo, ovov};
    g_prof_valid = false;
    g_launches = 0;
    if (int rc = dispatch_batches(P, in, ws, st, trip, e_trip, (size_t)P.T)) return rc;
    total_kernel<<<1, 256, 0, st>>>(e_trip, P.T, d_res);
    CU_TRY(cudaGetLastError());
    ++g_launches;
    if (e_triplet_out)
        CU_TRY(cudaMemcpyAsync(e_triplet_out, e_trip, (size_t)P.T * 3 * sizeof(double), cudaMemcpyDeviceToDevice, st));
    CU_TRY(cudaMemcpyAsync(e_out, d_res, 3 * sizeof(double), cudaMemcpyDeviceToHost, st));
    CU_TRY(cudaStreamSynchronize(st));
    return TRIPLES_OK;
}

int triples_energy_host(int nocc, int nvirt, const double* eps_o, const double* eps_v, const double* t1,
                        const double* t2, const double* vvvo, const double* ovoo, const double* ovov, int precision,
                        void* workspace, size_t workspace_bytes, void* cuda_stream, double* e_out,
                        double* e_triplet_out) {
    Plan P;
    const void* ptrs[8] = {eps_o, eps_v, t1, t2, vvvo, ovoo, ovov, e_out};
    if (int rc = validate_common(nocc, nvirt, precision, ptrs, 8, workspace, workspace_bytes, 0, P)) return rc;
    if (workspace_bytes < P.total_host)
        return fail(TRIPLES_EWORKSPACE, "workspace too small: %zu bytes given, %zu needed", workspace_bytes, P.total_host);
    if (int rc = check_device()) return rc;
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

int triples_energy_subset(int nocc, int nvirt, const double* eps_o, const double* eps_v, const double* t1,
                          const double* t2, const double* vvvo, const double* ovoo, const double* ovov, int precision,
                          int ntrip, const int* ijk, void* workspace, size_t workspace_bytes, void* cuda_stream,
                          double* e_out) {
    Plan P;
    const void* ptrs[7] = {eps_o, eps_v, t1, t2, vvvo, ovoo, ovov};
    if (int rc = validate_common(nocc, nvirt, precision, ptrs, 7, workspace, workspace_bytes, 0, P)) return rc;
    if (ntrip < 0 || (ntrip > 0 && (!ijk || !e_out))) return fail(TRIPLES_EINVAL, "bad triplet list");
    if ((long long)ntrip > P.T) return fail(TRIPLES_EINVAL, "more triplets (%d) than the restricted loop has (%lld)", ntrip, P.T);
    for (int n = 0; n < 7; ++n)
        if (misaligned(ptrs[n])) return fail(TRIPLES_EINVAL, "input pointer #%d is not 16-byte aligned", n);
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
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    uint8_t* ws = static_cast<uint8_t*>(workspace);
    double* e_trip = reinterpret_cast<double*>(ws + P.off_etrip);
    Inputs in{eps_o, eps_v, t1, t2, vvvo, ovoo, ovov};
    g_prof_valid = false;
    g_launches = 0;
    if (int rc = dispatch_batches(P, in, ws, st, trip, e_trip, (size_t)ntrip)) return rc;
    CU_TRY(cudaMemcpyAsync(e_out, e_trip, (size_t)ntrip * 3 * sizeof(double), cudaMemcpyDeviceToHost, st));
    CU_TRY(cudaStreamSynchronize(st));
    return TRIPLES_OK;
}

int triples_w_block(int nocc, int nvirt, const double* t2, const double* vvvo, const double* ovoo, int precision,
                    int i, int j, int k, void* workspace, size_t workspace_bytes, void* cuda_stream, double* W_out) {
    Plan P;
    const void* ptrs[4] = {t2, vvvo, ovoo, W_out};
    if (int rc = validate_common(nocc, nvirt, precision, ptrs, 4, workspace, workspace_bytes, 0, P)) return rc;
    if (i < 0 || j < 0 || k < 0 || i >= nocc || j >= nocc || k >= nocc) return fail(TRIPLES_EINVAL, "occupied index out of range");
    for (int n = 0; n < 3; ++n)
        if (misaligned(ptrs[n])) return fail(TRIPLES_EINVAL, "input pointer #%d is not 16-byte aligned", n);
    if (workspace_bytes < P.total)
        return fail(TRIPLES_EWORKSPACE, "workspace too small: %zu bytes given, %zu needed", workspace_bytes, P.total);
    if (int rc = check_device()) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    uint8_t* ws = static_cast<uint8_t*>(workspace);
    Operands op = carve_operands(P, ws);
    g_launches = 0;
    if (int rc = run_prepare(P, t2, vvvo, ovoo, op, st)) return rc;
    Maps maps;
    if (int rc = build_maps(P, op, &maps)) return rc;
    uint8_t* ubase = ws + P.off_u;
    const size_t ub = (size_t)UBLK * P.esz;   // U1, U2, U3 blocks of a tile are adjacent
    GemmJob gj[3] = {{i, j, k, 0, ubase, nullptr, 1, {0, 0, 0}},          // three groups of one job
                     {j, i, k, 1, ubase + ub, nullptr, 1, {0, 0, 0}},
                     {k, i, j, 2, ubase + 2 * ub, nullptr, 1, {0, 0, 0}}};
    GemmJob* d_gj = reinterpret_cast<GemmJob*>(ws + P.off_gjobs);
    CU_TRY(cudaMemcpyAsync(d_gj, gj, sizeof gj, cudaMemcpyHostToDevice, st));
    if (int rc = launch_gemm(P, maps, op, d_gj, 3, st)) return rc;
    if (precision == TRIPLES_FP64)
        assemble_w_kernel<double><<<kNumSM * 4, 256, 0, st>>>((const double*)ubase, nvirt, P.nt, W_out);
    else
        assemble_w_kernel<float><<<kNumSM * 4, 256, 0, st>>>((const float*)ubase, nvirt, P.nt, W_out);
    CU_TRY(cudaGetLastError());
    ++g_launches;
    CU_TRY(cudaStreamSynchronize(st));
    return TRIPLES_OK;
}

}  // extern "C"
