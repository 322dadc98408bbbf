/*
 * triples_b200.h -- C ABI of the B200 (sm_100a) closed-shell CCSD(T) perturbative triples energy.
 *
 * What it computes (arXiv:1609.08094, section 2.2):
 *
 *   Eq. (2.2.2), L94 : t_ijk^abc eps_ijk^abc = -P_ijk^abc [ sum_d t_ij^ad g_ckbd - sum_l t_il^ab g_cklj ]
 *   Eq. (2.2.3), L99 : P x_ijk^abc = x_ijk^abc + x_ikj^acb + x_jik^bac + x_jki^bca + x_kij^cab + x_kji^cba
 *   Eq. (2.2.4): z_ijk^abc eps_ijk^abc = -( t_i^a g_jbkc + t_j^b g_iakc + t_k^c g_iajb )
 *   Eq. (2.2.5): x~^abc = 2 ( 2/3 x^abc - x^acb + 1/3 x^bca )
 *   Eq. (2.2.1), L87 : E[4] = sum t~ t eps,  E[5] = sum z~ t eps,  E(T) = E[4] + E[5]
 *
 * evaluated over the restricted occupied triplets i<=j<=k (L119; task count Eq. (5.0.7b))
 * with the readings of DESIGN.md ("Readings"): D = eps_i+eps_j+eps_k-eps_a-eps_b-eps_c (< 0),
 *   W^abc  = numerator of Eq. (2.2.2) after P,   Vd^abc = numerator of Eq. (2.2.4),
 *   e_ijk  = sum_abc Z[W]^abc (W + Vd)^abc / D^abc,
 *   Z[W]^abc = 4W^abc + W^bca + W^cab - 2W^acb - 2W^cba - 2W^bac,
 *   E(T)   = sum_{i<=j<=k} (2 - delta_ij - delta_jk) e_ijk           (so E(T) < 0).
 *
 * Conventions for every entry point
 *   - Tensors are dense, row-major (C order), last index fastest, float64, no padding.
 *     Mulliken integrals (L63): vvvo[a][b][c][k] = (ab|ck), ovoo[i][a][j][k] = (ia|jk),
 *     ovov[i][a][j][b] = (ia|jb); t1[i][a] = t_i^a; t2[i][j][a][b] = t_ij^ab.
 *     Preconditions (not checked on the hot path): real orbitals (8-fold integral symmetry),
 *     t2[i][j][a][b] == t2[j][i][b][a], every D != 0.
 *   - "device" pointers are CUDA device pointers on the current device, 16-byte aligned;
 *     "host" pointers are ordinary host memory.  All pointers are caller-owned; inputs are
 *     never modified or freed.  The library allocates no device memory: all scratch comes from
 *     `workspace` (device, caller-owned, e.g. a torch.uint8 tensor), 256-byte aligned.
 *   - Work is enqueued on `cuda_stream` (a cudaStream_t, may be NULL for the default stream);
 *     the call synchronises that stream once before writing host outputs.
 *   - The only state the library owns -- the copy stream of streamed runs and the CUDA events of profiled /
 *     streamed runs -- is kept per device and per host thread: one host thread may use several GPUs in turn
 *     (cudaSetDevice before the call).  A streamed run that fails drains its copy stream before it returns.
 *   - Errors: a triples_status_t is returned, nothing aborts or throws; a message for the last
 *     non-OK status of the calling thread is available from triples_last_error().
 *     There is no CPU fallback: on a device that is not compute capability 10.x the compute
 *     entry points return TRIPLES_EARCH.
 *   - Device pointers are validated with cudaPointerGetAttributes: a host pointer where a device pointer is
 *     expected returns TRIPLES_EINVAL (it does not surface as a CUDA fault later).
 *   - precision: TRIPLES_FP64  = contractions in FP64 (DMMA), everything FP64;
 *                TRIPLES_MIXED = the paper's mixed precision (L125, L156): only the W build
 *                (the contractions) in single precision (operands scaled by a power of two and split
 *                x = h + l in FP16, h*h' + h*l' + l*h' on tcgen05 with FP32 accumulation, W stored FP32:
 *                W within 1e-6 of FP64 on the scale of W); Vd, D, the energy reduction and sums in FP64.
 *                TRIPLES_EMU64 = FP64-class contractions emulated on the INT8 tensor cores (a
 *                third point of the paper's precision study, L125, L156-L158): operands as 47-bit fixed point relative
 *                to the largest element of their tensor class (integrals / amplitudes), cut into six base-256
 *                digits; the digit products are exact integer GEMMs (tcgen05 kind::i8), recombined in FP64; W stored
 *                FP64, everything else as TRIPLES_FP64.  Tolerance: the FP64 one.  Error model: ABSOLUTE, ~2^-46 of
 *                the class maximum per operand element (an element 2^-n below the maximum keeps 47-n bits).
 *                Every entry point takes it (streamed / RI slices are staged in FP64 and digitised on the device).
 *                Measured on integrals that are NOT flat (synth decay option: B[Q,p,q] exp(-decay |p-q|), (vv|vo)
 *                spanning 1e12 and more, per-triplet energies spanning 4e5 .. 6e9): E(T), E[4], E[5] stay within
 *                6e-13 / 4e-13 / 3e-12 (EMU64) and 3e-7 (MIXED) of the oracle, and every per-triplet energy within
 *                3e-12 (EMU64) / 2e-7 (MIXED) of the LARGEST per-triplet energy; relative to ITS OWN size a triplet
 *                that is n orders of magnitude below the largest loses about n digits (EMU64: 1e-8 at a spread of 4e5,
 *                1.5e-5 at 6e9) -- one power-of-two scale per tensor class, not per slice or row.
 */
#ifndef TRIPLES_B200_H
#define TRIPLES_B200_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum { TRIPLES_FP64 = 0, TRIPLES_MIXED = 1, TRIPLES_EMU64 = 2 } triples_precision_t;

typedef enum {
    TRIPLES_OK = 0,
    TRIPLES_EINVAL = 1,      /* bad size, null or misaligned pointer, unknown precision, bad triplet */
    TRIPLES_EWORKSPACE = 2,  /* workspace too small: re-query triples_workspace_bytes */
    TRIPLES_ECUDA = 3,       /* a CUDA call failed; text in triples_last_error() */
    TRIPLES_EARCH = 4        /* device is not compute capability 10.x */
} triples_status_t;

/* Number of restricted triplets T = nocc(nocc+1)(nocc+2)/6 (Eq. (5.0.7b)); 0 if nocc < 1. */
long long triples_triplet_count(int nocc);

/* Enumeration order of the restricted loop: for i in [0,o): for j in [i,o): for k in [j,o).
 * ijk_out: host, 3*T ints.  This is the index order of e_triplet_out below. */
int triples_triplet_list(int nocc, int* ijk_out);

/* Bytes of device workspace triples_energy needs for (nocc, nvirt, precision); 0 on invalid
 * arguments.  Host-only computation, no CUDA call. */
size_t triples_workspace_bytes(int nocc, int nvirt, int precision);

/* Same for triples_energy_host (adds room for device copies of the seven inputs). */
size_t triples_workspace_bytes_host(int nocc, int nvirt, int precision);

/*
 * E(T) of Eq. (2.2.1)-(2.2.5) with all inputs resident on the device.
 *   eps_o[nocc], eps_v[nvirt], t1, t2, vvvo, ovoo, ovov : device, float64 (layouts above)
 *   e_out          : host, 3 doubles: e_out[0] = E(T), e_out[1] = E[4], e_out[2] = E[5]
 *   e_triplet_out  : device, 3*T doubles or NULL: for triplet n of triples_triplet_list,
 *                    [3n+0] = w*(e4+e5), [3n+1] = w*e4, [3n+2] = w*e5, w = 2-d_ij-d_jk
 * All sums are taken in a fixed order (no atomics): results are run-to-run bitwise identical.
 */
int triples_energy(int nocc, int nvirt,
                   const double* eps_o, const double* eps_v, const double* t1, const double* t2,
                   const double* vvvo, const double* ovoo, const double* ovov,
                   int precision,
                   void* workspace, size_t workspace_bytes, void* cuda_stream,
                   double* e_out, double* e_triplet_out);

/*
 * Same computation with all seven inputs in HOST memory (pinned or pageable): the library copies
 * them into `workspace` (device) on `cuda_stream`, runs triples_energy, and copies the results
 * back.  e_out: host, 3 doubles; e_triplet_out: HOST, 3*T doubles or NULL.
 */
int triples_energy_host(int nocc, int nvirt,
                        const double* eps_o, const double* eps_v, const double* t1, const double* t2,
                        const double* vvvo, const double* ovoo, const double* ovov,
                        int precision,
                        void* workspace, size_t workspace_bytes, void* cuda_stream,
                        double* e_out, double* e_triplet_out);

/*
 * triples_energy for callers that have no device memory to give and no way to get any.
 *
 * Who that is: every other compute entry point takes a caller-allocated `workspace`, which presumes the caller can
 * call cudaMalloc (or owns a pool).  Some cannot: a plug-in inside a host program (typically a quantum-chemistry
 * package, the setting of PAPER.md L228: the canonical (T) kernel run once per small fragment) whose own memory
 * manager has already claimed the device and hands plug-ins no allocator; code in a section that must not stall,
 * because cudaMalloc / cudaFree synchronise the whole device and can fail late when memory is fragmented; code
 * that runs under a rule "no allocation after start-up".  For them this entry point brings its scratch memory
 * along: a fixed array of TRIPLES_NOALLOC_SCRATCH_BYTES that is part of the library's device image.  The call
 * performs no cudaMalloc, cudaFree, stream / event creation or other allocating CUDA routine (profiling, which
 * would create events, is off for its duration); the caller passes only inputs and outputs.
 *
 * Same arguments, results and kernels as triples_energy (Eq. (2.2.1)-(2.2.5)) minus the workspace pair.  The
 * restricted loop is cut into narrower occupied-index windows (fewer triplets in flight) until the scratch the run
 * needs fits the array; per-triplet arithmetic does not depend on that width.
 *
 *   Limit  : the array is 32 MiB, a deliberately modest figure because EVERY GPU on which this library's device
 *            code gets loaded holds it until the process exits, used or not.  It is enough for fragment-sized
 *            problems, roughly nocc <= 8 with nvirt <= 40 (BASELINE.json configs[0]) in all three precisions;
 *            the need grows like 2 nocc nvirt^3 operand words.  A larger problem is refused before any GPU work
 *            with TRIPLES_EWORKSPACE and a message naming both byte counts; such a problem needs triples_energy
 *            and a real workspace.
 *   Set-up : the first call on each device looks the array's device address up (cudaGetSymbolAddress, with that
 *            device current; a failure is returned as TRIPLES_ECUDA) and keeps it.  That look-up may make the CUDA
 *            runtime load the library's device code, which is not permitted while a stream is being captured: make
 *            the first call on a device outside any stream capture.
 *   Sharing: there is one array per device, shared by every call, thread and stream of the process.  A call
 *            first zeroes the part it is going to use, so it never sees what an earlier call left behind, and
 *            it returns after synchronising its stream.  Two calls that overlap in time on the same GPU (from
 *            two host threads, or on two streams) write the same memory and race: results are then undefined.
 *            Serialise them.
 */
#define TRIPLES_NOALLOC_SCRATCH_BYTES (32u << 20)
int triples_energy_noalloc(int nocc, int nvirt,
                           const double* eps_o, const double* eps_v, const double* t1, const double* t2,
                           const double* vvvo, const double* ovoo, const double* ovov,
                           int precision, void* cuda_stream,
                           double* e_out, double* e_triplet_out);

/*
 * Triplet-sharded run ("each loop cycle is data independent ... trivially
 * distributed", L121, L206): the batches (window blocks) of the restricted loop are cut into `nshards` contiguous
 * ranges of equal contraction-job count (triples_plan_shards); this call computes range `shard` only.
 * Inputs are replicated.  e_out = this shard's partial (E(T), E[4], E[5]); the caller adds the partials of all
 * shards in shard order (three doubles per rank -- the only exchange step).  e_triplet_out rows of other shards
 * are zero.  triples_energy is the case shard = 0, nshards = 1.
 */
int triples_energy_sharded(int nocc, int nvirt,
                           const double* eps_o, const double* eps_v, const double* t1, const double* t2,
                           const double* vvvo, const double* ovoo, const double* ovov,
                           int precision, int shard, int nshards,
                           void* workspace, size_t workspace_bytes, void* cuda_stream,
                           double* e_out, double* e_triplet_out);

/* Host-side view of that partition: shard_of_triplet (host, T ints or NULL; -1 for i=j=k), jobs_per_shard (host,
 * nshards long longs or NULL).  Returns the number of batches or -1 on invalid arguments. */
long long triples_plan_shards(int nocc, int nvirt, int precision, int nshards, int* shard_of_triplet,
                              long long* jobs_per_shard);

/*
 * Out-of-core run ("tiles of t2 and ERIs transferred asynchronously, pinned
 * memory"; L216, L220: sizes "as large as allowed by host memory").  The (vv|vo) integrals stay in HOST memory,
 * slice-major:   vovv_host[k][a][b][c] = (ab|ck)   (nocc slices of nvirt^3 doubles, pinned for full copy speed);
 * every other input is device-resident as in triples_energy.  The device keeps a cache of repacked slices X_r
 * (+ XT_r): as many slots as `workspace_bytes` allows (triples_cache_slots), at least the slices of two
 * consecutive batches.  A batch is a block of occupied-index windows of width `win` <= 4; a small budget is met
 * by a narrower window (fewer U buffers, 6 win slices minimum): the call takes the widest window whose minimum
 * fits, then the largest cache.  Which slice sits in which slot when is planned
 * on the host for the whole launch order (Belady replacement, triples_plan_slices); the copies of batch b+2 run
 * on a library-owned copy stream while batch b+1 computes.  Same kernels and the same batches as triples_energy:
 * per-triplet energies are bitwise identical to the resident run.
 *   vvvo_absmax : TRIPLES_MIXED and TRIPLES_EMU64 (ignored by TRIPLES_FP64): the largest |(ab|ck)| if the caller
 *                 knows it (it fixes the power-of-two operand scale of the packed operands); <= 0: the library scans
 *                 the host tensor once (one extra pass of copies).  A value ABOVE the true maximum only costs
 *                 precision (one bit per factor of two).  A value BELOW it would overflow FP16 (mixed) or wrap the
 *                 top base-256 digit (emulated FP64): the repack detects any element beyond the bound the value
 *                 implies and the call returns TRIPLES_EINVAL instead of wrong energies (e_out is then invalid).
 */
int triples_energy_streamed(int nocc, int nvirt,
                            const double* eps_o, const double* eps_v, const double* t1, const double* t2,
                            const double* vovv_host, const double* ovoo, const double* ovov,
                            int precision, double vvvo_absmax,
                            void* workspace, size_t workspace_bytes, void* cuda_stream,
                            double* e_out, double* e_triplet_out);

/* Workspace bytes of triples_energy_streamed with a slice cache of `nslots` slots (clamped to [minimum, nocc];
 * nslots <= 0: the minimum) and windows of width <= `win` (win <= 0: the default of the resident run).
 * 0 on invalid arguments. */
size_t triples_workspace_bytes_streamed(int nocc, int nvirt, int precision, int nslots, int win);

/*
 * RI-direct run (Eq. (2.1.3): (pq|rs) = sum_Q B[Q,p,q] B[Q,r,s]).
 * The vvvo tensor is never materialised: a slice X_r[d,b,c] = sum_Q B[Q,d,b] B[Q,c,r] is rebuilt on the device
 * by an FP64 DMMA GEMM (M = v^2, N = v, K = naux) whenever a batch needs it and the slice cache does not hold it.
 *   B : device, [naux][n][n] doubles, n = nocc + nvirt, occupied orbitals first, symmetric in the orbital pair.
 * ovoo / ovov / t2 are passed as for triples_energy.  Extra work: 2 naux v^3 flop per slice built
 * (triples_last_profile out[11], out[13]); with a cache of nocc slots every slice is built once.
 * TRIPLES_MIXED: slices are built in FP64 and split-packed; the operand scale comes from the Cauchy-Schwarz bound
 * |(ab|ck)| <= |B[:,a,b]| |B[:,c,k]|.
 */
int triples_energy_ri(int nocc, int nvirt, int naux,
                      const double* eps_o, const double* eps_v, const double* t1, const double* t2,
                      const double* B, const double* ovoo, const double* ovov,
                      int precision,
                      void* workspace, size_t workspace_bytes, void* cuda_stream,
                      double* e_out, double* e_triplet_out);

size_t triples_workspace_bytes_ri(int nocc, int nvirt, int naux, int precision, int nslots, int win);

/* Slice-cache slots a workspace of `workspace_bytes` gives (mode 1 = streamed, 2 = RI; naux: RI only) and, in
 * *win_out (host or NULL), the window width the run will use; 0 if not even window 1 fits. */
int triples_cache_slots(int nocc, int nvirt, int naux, int precision, int mode, size_t workspace_bytes, int* win_out);

/*
 * Host-side plan of the slice cache (pure host arithmetic): for the full restricted loop, a cache of `nslots`
 * slots and windows of width <= `win` (both clamped as above) in `mode` (1 = streamed: a batch's loads may not
 * evict what the previous batch uses; 2 = RI), which slice is loaded into which slot before which batch.
 *   loads_out : host, 3*loads_cap ints or NULL: {batch, r, slot} per load, in order
 *   jobs_out  : host, 5*jobs_cap ints or NULL: per contraction job in launch order
 *               {batch, q, r, cache slot of XT_q, cache slot of X_r}
 *   info_out  : host, 4 ints or NULL: {slots used, window width, batches, jobs}
 * Returns the number of loads, or -1 on error.
 */
long long triples_plan_slices(int nocc, int nvirt, int precision, int mode, int nslots, int win, int* loads_out,
                              long long loads_cap, int* jobs_out, long long jobs_cap, int* info_out);

/*
 * Per-triplet energies of a caller-chosen list of restricted triplets (the sampled-parity
 * protocol for the configurations whose full oracle run is out of reach).
 *   ntrip, ijk (host, 3*ntrip ints, each 0 <= i <= j <= k < nocc)
 *   e_out: host, 3*ntrip doubles, layout as e_triplet_out above (weighted).
 * Workspace requirement: triples_workspace_bytes.
 */
int triples_energy_subset(int nocc, int nvirt,
                          const double* eps_o, const double* eps_v, const double* t1, const double* t2,
                          const double* vvvo, const double* ovoo, const double* ovov,
                          int precision, int ntrip, const int* ijk,
                          void* workspace, size_t workspace_bytes, void* cuda_stream,
                          double* e_out);

/*
 * W_ijk^abc = P_ijk^abc [ sum_d t_ij^ad g_ckbd - sum_l t_il^ab g_cklj ]  (Eq. (2.2.2)-(2.2.3))
 * for ONE ordered (i,j,k), any order, written as float64 W_out[a][b][c] (device, nvirt^3 doubles).
 * Runs the same contraction kernels as triples_energy (in `precision`) followed by the
 * permutation-accumulate; meant for elementwise parity tests of the contraction stage.
 */
int triples_w_block(int nocc, int nvirt,
                    const double* t2, const double* vvvo, const double* ovoo,
                    int precision, int i, int j, int k,
                    void* workspace, size_t workspace_bytes, void* cuda_stream,
                    double* W_out);

/*
 * Timing of the calling thread's last triples_energy / _host / _subset call, measured with CUDA
 * events on `cuda_stream` when profiling was switched on with triples_set_profiling(1) before it.
 *   out[0] prepare (repack) ms          out[1] contraction kernels, summed ms
 *   out[2] contraction launches         out[3] fused reduction kernels, summed ms
 *   out[4] reduction launches           out[5] other kernels (finalize/sum), summed ms
 *   out[6] other launches               out[7] contraction flops executed (12v^4+12ov^3 per
 *                                              triplet, coinciding terms of i=j / j=k computed once)
 *   out[8] reduction algorithmic bytes  out[9] triplets executed (i=j=k skipped)
 *   out[10] per-batch slice work, summed ms (streamed: repack of arrived slices; RI: slice GEMMs + repack)
 *   out[11] slices loaded / built       out[12] host->device bytes of streamed slices
 *   out[13] flops of the RI slice GEMMs out[14..15] reserved (0)
 * Returns TRIPLES_EINVAL if no profiled call has happened.
 */
int triples_last_profile(double* out16);
void triples_set_profiling(int on);

/*
 * Host-side planner (S1; Eq. (5.0.7b)): how triples_energy cuts the restricted loop into
 * launches. Pure host arithmetic, no GPU needed. A batch is the set of restricted triplets of one block
 * I x J x K of occupied-index windows; inside a batch the contraction jobs G(p,q,r) are sorted by (q,r)
 * and the jobs sharing (q,r) -- the same (vv|vo) slices -- form a group that the kernels walk together.
 *   batch_of_triplet : host, T ints or NULL: batch of triplet n of triples_triplet_list (-1 for i=j=k,
 *                      which contributes exactly zero and is skipped)
 *   jobs_out         : host, 3*T*6 ints or NULL: per job, in launch order,
 *                      {batch, p, q, r, first job of its group (relative to the batch), group size}
 *   njobs_out        : host or NULL: number of jobs (<= 3*T; a triplet with i=j or j=k has two)
 * Returns the number of batches, or -1 on invalid sizes / precision (message in triples_last_error).
 */
long long triples_plan_batches(int nocc, int nvirt, int precision, int* batch_of_triplet, int* jobs_out,
                               long long* njobs_out);

/*
 * FP64 tensor-core (mma.sync.m8n8k4.f64, DMMA) peak of the current device in TFLOP/s: a register-resident DMMA
 * loop on every SM, best of three timed repetitions of `iters` iterations (CUDA events on `cuda_stream`).  This is
 * the roofline denominator of the FP64 contraction kernel, measured in the process that measures the numerator.
 * workspace: device, at least 148*256*8 bytes.
 */
int triples_probe_fp64_peak(void* workspace, size_t workspace_bytes, void* cuda_stream, int iters, double* tflops_out);

/*
 * tcgen05.mma peak of the current device for the two instruction kinds the packed contractions use, in Tera-operations
 * per second (2 x multiply-adds): kind 0 = kind::f16 (FP16 x FP16 -> FP32, M = 256 over a CTA pair, N = 256, K = 16; the
 * TRIPLES_MIXED contraction spends three of these per FP32-class product), kind 1 = kind::i8 (S8 x S8 -> S32, N = 80,
 * K = 32; TRIPLES_EMU64 spends 21 per FP64-class product).  An issue loop on operands resident in shared memory with
 * TMEM accumulators and no global traffic, on every co-resident CTA pair, for about `seconds` (a short run gives the
 * burst figure, ~2 s the figure under the power cap).  *sm_mhz_out (host or NULL): the SM clock during the loop, from
 * clock64 / globaltimer inside the kernel.  These are the roofline denominators of the two tcgen05 contraction
 * kernels (the precision study; SURVEY 8(d) "to be measured").
 * workspace: device, at least 148*8 bytes.
 */
int triples_probe_tc_peak(int kind, double seconds, void* workspace, size_t workspace_bytes, void* cuda_stream,
                          double* tops_out, double* sm_mhz_out);

/* Number of CUDA kernels the calling thread's last compute call (triples_energy / _host / _subset / _w_block)
 * launched (repack + contraction + reduction + finalize + total). */
long long triples_last_launch_count(void);

/* Thread-local message for the last non-OK status ("" if none). Never NULL. */
const char* triples_last_error(void);

/* ABI version of this header (integer, bumped on any signature change). */
int triples_abi_version(void);

#ifdef __cplusplus
}
#endif
#endif /* TRIPLES_B200_H */
