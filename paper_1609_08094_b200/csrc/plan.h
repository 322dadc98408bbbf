// plan.h -- host-side planner (S1 of DESIGN.md): triplet enumeration, tile-orbit table, batching, workspace layout.
// Pure host arithmetic (no CUDA calls) so that the CPU test-suite can exercise it through the C ABI.
#pragma once
#include <cstddef>
#include <algorithm>
#include <cstdint>
#include <cstdlib>
#include <vector>

namespace tb {

constexpr int kMaxVirt = 2040;   // tile indices of the 8-wide reduction tiles fit a byte
constexpr int kMaxOcc = 1024;
constexpr int kNumSM = 148;
constexpr int kRedWarps = 8;     // consumer warps of the fused reduction: one partial per (triplet, orbit, warp)

struct Triplet { int i, j, k; long long index; };   // index = position in the i<=j<=k enumeration

inline long long triplet_count(int o) { return o < 1 ? 0 : (long long)o * (o + 1) * (o + 2) / 6; }

// Enumeration order of the restricted loop (count Eq. (5.0.7b)).
inline void enumerate_triplets(int o, std::vector<Triplet>& out) {
    out.clear();
    long long n = 0;
    for (int i = 0; i < o; ++i)
        for (int j = i; j < o; ++j)
            for (int k = j; k < o; ++k) out.push_back({i, j, k, n++});
}

// Position of (i<=j<=k) in that enumeration, closed form.
inline long long triplet_index(int o, int i, int j, int k) {
    // triplets with first index < i: sum_{x<i} (o-x)(o-x+1)/2 = T(o) - T(o-i)
    auto T3 = [](long long n) { return n * (n + 1) * (n + 2) / 6; };
    auto T2 = [](long long n) { return n * (n + 1) / 2; };
    const long long m = o - i;                     // j,k range over [i,o): m values
    return T3(o) - T3(m) + (T2(m) - T2(m - (j - i))) + (k - j);
}

// Weight of a restricted triplet (Q4): 2 - delta_ij - delta_jk.
inline double triplet_weight(int i, int j, int k) { return 2.0 - (i == j ? 1.0 : 0.0) - (j == k ? 1.0 : 0.0); }

struct Orbit { uint8_t A, B, C, sym; };   // tiles A<=B<=C of the virtual cube; sym = |stabiliser| in {1,2,6}

inline int num_red_tiles(int v) { return (v + 7) / 8; }
inline long long orbit_count(int v) { const long long n = num_red_tiles(v); return n * (n + 1) * (n + 2) / 6; }
inline void enumerate_orbits(int v, std::vector<Orbit>& out) {
    out.clear();
    const int n = num_red_tiles(v);
    for (int A = 0; A < n; ++A)
        for (int B = A; B < n; ++B)
            for (int C = B; C < n; ++C) {
                const int sym = (A == B && B == C) ? 6 : ((A == B || B == C) ? 2 : 1);
                out.push_back({(uint8_t)A, (uint8_t)B, (uint8_t)C, (uint8_t)sym});
            }
}

enum GemmCfgId { CFG_M120_N128 = 0, CFG_M80_N192 = 1, CFG_M40_N256 = 2 };

// CTAs per MMA tile of the mixed contraction: a CTA pair (cta_group::2, gemm_f16split.cuh)
inline int tf_cluster_size() { return 2; }

// Where the (vv|vo) slices X_r come from
enum SliceMode {
    SLICES_RESIDENT = 0,   // the caller's vvvo tensor is on the device: every slice is repacked once, slot = r
    SLICES_STREAMED = 1,   // slices live in host memory [r][a][b][c]; a device cache of nslots slots, prefetched
    SLICES_RI = 2          // slices are rebuilt on the device from the RI factors B[Q][p][q] when a batch needs them
};

struct Plan {
    int o = 0, v = 0, vp = 0, op = 0, prec = 0;
    int vk = 0, ok = 0;         // mixed path: K pitches (4-byte words) of the packed K-major operands (v, o rounded up to 32)
    int mode = SLICES_RESIDENT; // SliceMode
    int nslots = 0;             // slots of the X / XT slice cache (resident: o)
    int naux = 0, nauxp = 0;    // RI mode: auxiliary functions, K pitch of the repacked factors
    int ri_cfg = 0, ri_BM = 0, ri_BN = 0, ri_mtiles = 0, ri_ntiles = 0;   // RI slice GEMM tiles
    int nstage = 0;             // FP64 staging slices (mixed streamed: 2 x 3 win; mixed RI: 1)
    size_t n_slice = 0;         // elements (FP64) / words (mixed) of one slot of X (or XT)
    size_t off_stage = 0, off_bt = 0, off_bo = 0, off_loads = 0;
    int cfg = 0, BM = 0, BN = 0, mtiles = 0, ntiles = 0;      // FP64 contraction tiles
    int tf_bn = 0, tf_ntiles = 0, tf_mtiles = 0;              // mixed contraction tiles: 128 (b,c) rows x tf_bn a-columns
    int tf_cs = 1, tf_npad = 0;                               // CTAs per MMA tile (2 = cta_group::2 pair); N-side rows a CTA stages
    int nb = 0;                 // triplets per batch (at most win^3)
    int win = 1;                // batch = block of occupied-index windows of this width (see make_plan)
    long long T = 0;            // restricted triplets
    int norb = 0, nt = 0;       // tile orbits, 8-wide tiles per virtual axis
    int red_gx = 0;             // CTA columns of the fused reduction (orbit stride), fixed by v
    size_t n_side = 0;          // doubles of one triplet's side buffer (reduce.cuh)
    size_t off_side = 0;
    size_t esz = 8;             // bytes per stored U element (FP64 / emulated FP64: 8, mixed: 4)
    size_t osz = 8;             // bytes per stored operand word (FP64: 8; mixed and emulated FP64: 4-byte packed words)
    int kchunks_v = 0, kchunks_o = 0;   // packed paths: 32-element K chunks a virtual / occupied operand row holds
    size_t n_x = 0, n_ot = 0, n_t2 = 0, n_u = 0;   // elements of one X (or XT), Ot, T2, one U buffer
    size_t n_t2k = 0;                              // mixed: elements of T2K (or T2KT)
    size_t off_t2k = 0, off_t2kt = 0;
    // workspace offsets (bytes)
    size_t off_x = 0, off_xt = 0, off_ot = 0, off_t2 = 0;
    size_t off_u = 0, off_part = 0, off_etrip = 0, off_result = 0, off_gjobs = 0, off_rjobs = 0, off_fjobs = 0,
           off_orb = 0;
    size_t total = 0;
    // host variant: device copies of the inputs follow
    size_t off_in[7] = {0, 0, 0, 0, 0, 0, 0};
    size_t in_bytes[7] = {0, 0, 0, 0, 0, 0, 0};
    size_t total_host = 0;
};

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// slots the slice cache needs at least: the slices of the batch that runs (3 windows) and, when slices are
// prefetched while the previous batch still computes (streamed), those of that batch as well
inline int min_slots(int o, int win, int mode) {
    const int n = (mode == SLICES_STREAMED ? 6 : 3) * win;
    return n < o ? n : o;
}

// Returns false on invalid sizes.  precision: 0 = FP64, 1 = MIXED.  nslots: slice-cache slots (streamed / RI; 0 = the
// minimum, clamped to [min_slots, o]); naux: RI mode only; win_cap > 0 limits the window width (a smaller window
// needs fewer U buffers and a smaller minimum cache: how a streamed / RI run fits a small device budget).
inline bool make_plan(int o, int v, int prec, Plan& P, int mode = SLICES_RESIDENT, int nslots = 0, int naux = 0,
                      int win_cap = 0) {
    if (o < 1 || v < 1 || o > kMaxOcc || v > kMaxVirt || (prec < 0 || prec > 2)) return false;
    if (mode < 0 || mode > 2 || nslots < 0 || (mode == SLICES_RI && naux < 1)) return false;
    P = Plan();
    P.o = o; P.v = v; P.prec = prec; P.mode = mode;
    P.vp = (v + 1) & ~1;
    P.op = (o + 1) & ~1;
    P.esz = prec == 1 ? 4 : 8;
    P.osz = prec == 0 ? 8 : 4;
    P.T = triplet_count(o);
    P.norb = (int)orbit_count(v);
    // CTA tile: the M tile (40, 80 or 120 rows) that wastes the fewest padded rows; ties -> larger tile
    const int bms[3] = {120, 80, 40};
    const int ids[3] = {CFG_M120_N128, CFG_M80_N192, CFG_M40_N256};
    const int bns[3] = {128, 192, 256};
    long long best = -1;
    for (int c = 0; c < 3; ++c) {
        const long long padded = (long long)((v + bms[c] - 1) / bms[c]) * bms[c];
        if (best < 0 || padded < best) { best = padded; P.cfg = ids[c]; P.BM = bms[c]; P.BN = bns[c]; }
    }
    const long long N = (long long)v * P.vp;
    P.mtiles = (v + P.BM - 1) / P.BM;
    P.ntiles = (int)((N + P.BN - 1) / P.BN);
    P.n_slice = (size_t)v * v * P.vp;
    P.n_ot = (size_t)o * o * v * P.op;
    P.n_t2 = (size_t)o * o * v * P.vp;
    P.nt = num_red_tiles(v);
    P.n_u = (size_t)P.nt * P.nt * P.nt * 512;          // blocked layout of ulayout.cuh
    P.n_side = (size_t)P.nt * P.nt * 448;             // tile-pair records of reduce.cuh
    if (prec != 0) {   // packed K-major operands, transposed tiles (gemm_f16split.cuh / gemm_emu64.cuh)
        if (prec == 1) {       // FP16 split: 32 words (one 128-byte row) per 32-wide K chunk
            P.vk = (v + 31) / 32 * 32; P.ok = (o + 31) / 32 * 32;
            P.kchunks_v = P.vk / 32; P.kchunks_o = P.ok / 32;
            P.tf_ntiles = (v + 255) / 256;
            P.tf_bn = (((v + P.tf_ntiles - 1) / P.tf_ntiles) + 15) & ~15;
        } else {               // emulated FP64: 96 words (three 128-byte rows of digit pairs) per 64-wide K chunk
            P.vk = (v + 63) / 64 * 96; P.ok = (o + 63) / 64 * 96;
            P.kchunks_v = P.vk / 96 * 2; P.kchunks_o = P.ok / 96 * 2;
            // tile width 80 / 64 / 48 columns: MMA time goes with the padded column count; the narrower tiles re-stage
            // the M-side rows more often (bytes per MMA clock 38 / 46 / 58 against the ~42 an SM can take in)
            const int bnc[3] = {80, 64, 48};
            const double feed[3] = {1.0, 1.09, 1.38};
            double bestc = -1.0;
            for (int c = 0; c < 3; ++c) {
                const double cost = (double)((v + bnc[c] - 1) / bnc[c] * bnc[c]) * feed[c];
                if (bestc < 0 || cost < bestc) { bestc = cost; P.tf_bn = bnc[c]; }
            }
            P.tf_ntiles = (v + P.tf_bn - 1) / P.tf_bn;
        }
        P.tf_mtiles = (int)((N + 127) / 128);
        // CTA pairs (cta_group::2): a pair owns two consecutive m-tiles, each CTA stages half of the N-side rows
        // (tf_bn is a multiple of 16, so a half is whole 8-row swizzle atoms)
        P.tf_cs = tf_cluster_size();
        P.tf_npad = P.tf_bn / P.tf_cs;
        P.n_slice = (size_t)v * P.vp * P.vk;
        P.n_t2 = (size_t)o * o * v * P.vk;
        P.n_ot = (size_t)o * o * v * P.ok;
        P.n_t2k = (size_t)o * v * P.vp * P.ok;
    }
    // Batch = all restricted triplets of one block I x J x K of occupied-index windows of width `win` (S1).  Inside
    // a block every contraction job (p; q,r) has win - 1 siblings with the same (q,r), i.e. the same X_r / XT_q
    // slices, which the contraction kernels walk tile by tile together: the big (vv|vo) operand then comes from HBM
    // once per group instead of once per job.  win: as wide as the U buffers allow (22 GiB cap,
    // sized for the 180 GB part next to 2 x 35 GB of repacked integrals at the largest config), at most 4.
    const long long cap = (long long)((22ULL << 30) / (3 * P.n_u * P.esz));
    int win = 1;
    while (win < 4 && win < o && (long long)(win + 1) * (win + 1) * (win + 1) <= cap && (win_cap <= 0 || win < win_cap)) ++win;
    P.win = win;
    long long nb = (long long)win * win * win;
    if (nb > P.T) nb = P.T;
    P.nb = (int)nb;
    if (mode == SLICES_RESIDENT) {
        P.nslots = o;
    } else {
        const int lo = min_slots(o, win, mode);
        P.nslots = nslots < lo ? lo : (nslots > o ? o : nslots);
    }
    P.n_x = (size_t)P.nslots * P.n_slice;
    if (prec != 0 && mode == SLICES_STREAMED) P.nstage = 2 * min_slots(o, win, SLICES_RI);   // packed paths: FP64 staging
    if (prec != 0 && mode == SLICES_RI) P.nstage = 1;
    if (mode == SLICES_RI) {   // X_r[(d,b)][c] = sum_Q Bt[(d,b)][Q] Bo[r][Q][c]: M = v^2, N = v, K = naux
        P.naux = naux;
        P.nauxp = (naux + 1) & ~1;
        long long bestn = -1;
        for (int c = 0; c < 3; ++c) {
            const long long padded = (long long)((v + bns[c] - 1) / bns[c]) * bns[c];
            if (bestn < 0 || padded < bestn) { bestn = padded; P.ri_cfg = ids[c]; P.ri_BM = bms[c]; P.ri_BN = bns[c]; }
        }
        P.ri_mtiles = (int)(((long long)v * v + P.ri_BM - 1) / P.ri_BM);
        P.ri_ntiles = (v + P.ri_BN - 1) / P.ri_BN;
    }

    size_t off = 0;
    auto take = [&](size_t bytes) { size_t at = off; off = align_up(off + bytes, 1024); return at; };
    P.off_x = take(P.n_x * P.osz);
    P.off_xt = take(P.n_x * P.osz);
    P.off_ot = take(P.n_ot * P.osz);
    P.off_t2 = take(P.n_t2 * P.osz);
    if (prec != 0) {   // occupied-segment M-side operands of the transposed GEMMs
        P.off_t2k = take(P.n_t2k * P.osz);
        P.off_t2kt = take(P.n_t2k * P.osz);
    }
    if (P.nstage) P.off_stage = take((size_t)P.nstage * v * v * P.vp * 8);
    if (mode == SLICES_RI) {
        P.off_bt = take((size_t)v * v * P.nauxp * 8);
        P.off_bo = take((size_t)o * naux * P.vp * 8);
    }
    P.off_u = take((size_t)P.nb * 3 * P.n_u * P.esz);
    P.red_gx = P.norb < kNumSM ? P.norb : kNumSM;
    P.off_part = take((size_t)P.nb * P.red_gx * kRedWarps * 16);
    P.off_side = take((size_t)P.nb * P.n_side * 8);
    P.off_etrip = take((size_t)P.T * 3 * 8);
    P.off_result = take(256);
    P.off_gjobs = take((size_t)P.T * 3 * 48);
    P.off_rjobs = take((size_t)P.T * 48);
    P.off_fjobs = take((size_t)P.T * 16);
    P.off_orb = take((size_t)P.norb * 4);
    if (mode == SLICES_RI) P.off_loads = take((size_t)P.T * 24 * 8 + 64);   // <= 3 win loads per batch, two tables
    P.total = off;
    if (mode == SLICES_RESIDENT) {
        const size_t in_elems[7] = {(size_t)o, (size_t)v, (size_t)o * v, (size_t)o * o * v * v, (size_t)v * v * v * o,
                                    (size_t)o * v * o * o, (size_t)o * v * o * v};
        for (int n = 0; n < 7; ++n) { P.in_bytes[n] = in_elems[n] * 8; P.off_in[n] = take(P.in_bytes[n]); }
    }
    P.total_host = off;
    return true;
}

// ------------------------------------------------------------------------------------------------ batches (S1)
// One contraction job G(p,q,r) of a batch.  u / u2: which of the triplet slot's three U
// buffers receive it (u2 = -1 unless a coinciding pair i=j or j=k makes one G serve two of them).
struct JobDesc { int p, q, r, slot, u, u2, gstart, gsize, xr, xq; };   // xr / xq: cache slots of X_r / XT_q

struct SliceLoad { int r, slot; };   // slice X_r (and XT_r) goes into this slot of the cache

struct BatchPlan {
    std::vector<Triplet> work;     // triplets in execution order (i=j=k dropped: they contribute exactly zero)
    std::vector<size_t> bstart;    // batch b = work[bstart[b] .. bstart[b+1]); slot of a triplet = offset in its batch
    std::vector<JobDesc> jobs;     // jobs of all batches; inside a batch sorted by (q,r,p)
    std::vector<int> jstart;       // batch b = jobs[jstart[b] .. jstart[b+1]); gstart is relative to jstart[b]
    double distinct_u = 0.0;       // U buffers the reductions read (2 per triplet with a coinciding pair, else 3)
    std::vector<SliceLoad> loads;  // streamed / RI: slices to bring into the cache, in batch order
    std::vector<int> lstart;       // batch b needs loads[lstart[b] .. lstart[b+1]) before its contraction starts
};

// Batches = the triplets of one block I x J x K of occupied-index windows of width P.win (at most P.nb each).
// Inside a batch the jobs with the same (q,r) -- the same X_r / XT_q operand slices -- form one group.
inline void build_batches(const Plan& P, const std::vector<Triplet>& trip, BatchPlan& B) {
    B = BatchPlan();
    for (const Triplet& t : trip)
        if (!(t.i == t.j && t.j == t.k)) B.work.push_back(t);
    const int win = P.win, nwin = (P.o + win - 1) / win;
    auto key = [&](const Triplet& t) { return ((long long)(t.i / win) * nwin + t.j / win) * nwin + t.k / win; };
    // stable: inside a block the enumeration order of the caller's list is kept
    std::vector<Triplet> sorted(B.work);
    std::vector<long long> keys(sorted.size());
    for (size_t n = 0; n < sorted.size(); ++n) keys[n] = key(sorted[n]);
    std::vector<size_t> order(sorted.size());
    for (size_t n = 0; n < order.size(); ++n) order[n] = n;
    std::stable_sort(order.begin(), order.end(), [&](size_t x, size_t y) { return keys[x] < keys[y]; });
    for (size_t n = 0; n < order.size(); ++n) B.work[n] = sorted[order[n]];
    const size_t nwork = B.work.size();
    for (size_t n = 0; n < nwork; ++n)
        if (n == 0 || key(B.work[n]) != key(B.work[n - 1]) || n - B.bstart.back() == (size_t)P.nb) B.bstart.push_back(n);
    B.bstart.push_back(nwork);
    const size_t nbatch = B.bstart.size() - 1;
    for (size_t b = 0; b < nbatch; ++b) {
        const size_t j0 = B.jobs.size();
        B.jstart.push_back((int)j0);
        for (size_t n = B.bstart[b]; n < B.bstart[b + 1]; ++n) {
            const Triplet& t = B.work[n];
            const int slot = (int)(n - B.bstart[b]);
            if (t.i == t.j) {            // G(j,i,k) = G(i,j,k): one job, two destinations
                B.jobs.push_back({t.i, t.j, t.k, slot, 0, 1, 0, 1, 0, 0});
                B.jobs.push_back({t.k, t.i, t.j, slot, 2, -1, 0, 1, 0, 0});
            } else if (t.j == t.k) {     // G(k,i,j) = G(j,i,k)
                B.jobs.push_back({t.i, t.j, t.k, slot, 0, -1, 0, 1, 0, 0});
                B.jobs.push_back({t.j, t.i, t.k, slot, 1, 2, 0, 1, 0, 0});
            } else {
                B.jobs.push_back({t.i, t.j, t.k, slot, 0, -1, 0, 1, 0, 0});   // U1 = G(i,j,k)[a][b][c]
                B.jobs.push_back({t.j, t.i, t.k, slot, 1, -1, 0, 1, 0, 0});   // U2 = G(j,i,k)[b][a][c]
                B.jobs.push_back({t.k, t.i, t.j, slot, 2, -1, 0, 1, 0, 0});   // U3 = G(k,i,j)[c][a][b]
            }
            B.distinct_u += 1.0 + (t.i != t.j) + (t.j != t.k);
        }
        std::sort(B.jobs.begin() + j0, B.jobs.end(), [](const JobDesc& x, const JobDesc& y) {
            return x.q != y.q ? x.q < y.q : (x.r != y.r ? x.r < y.r : (x.p != y.p ? x.p < y.p : x.slot < y.slot));
        });
        for (size_t g = j0; g < B.jobs.size();) {
            size_t e = g;
            while (e < B.jobs.size() && B.jobs[e].q == B.jobs[g].q && B.jobs[e].r == B.jobs[g].r) ++e;
            for (size_t x = g; x < e; ++x) {
                B.jobs[x].gstart = (int)(g - j0); B.jobs[x].gsize = (int)(e - g);
                B.jobs[x].xr = B.jobs[x].r; B.jobs[x].xq = B.jobs[x].q;       // resident: slot = slice
            }
            g = e;
        }
    }
    B.jstart.push_back((int)B.jobs.size());
}


// ------------------------------------------------------------------------------------------------ sharding (NEXT-3)
// Static partition of the batches (window blocks) over nshards ranks ("trivially distributed", L121):
// contiguous ranges of the launch order -- consecutive window blocks share (vv|vo) slices -- balanced by contraction
// job count (every job costs the same 4v^3(v+o) flop, L198-L206).  Keeps the batches [b0, b1) of `shard`.
inline void shard_range(const BatchPlan& B, int shard, int nshards, size_t& b0, size_t& b1) {
    const size_t nbatch = B.bstart.size() - 1;
    const long long njobs = (long long)B.jobs.size();
    auto cut = [&](int s) -> size_t {      // the batch boundary nearest to the s-th equal share of the jobs
        if (s <= 0) return 0;
        if (s >= nshards) return nbatch;
        const long long target = njobs * s / nshards;
        size_t b = 0;
        while (b < nbatch && B.jstart[b] < target) ++b;
        if (b > 0 && target - B.jstart[b - 1] < B.jstart[b] - target) --b;
        return b;
    };
    b0 = cut(shard);
    b1 = cut(shard + 1);
}

inline void select_shard(BatchPlan& B, int shard, int nshards) {
    if (nshards <= 1) return;
    size_t b0, b1;
    shard_range(B, shard, nshards, b0, b1);
    BatchPlan S;
    S.bstart.push_back(0);
    for (size_t b = b0; b < b1; ++b) {
        S.jstart.push_back((int)S.jobs.size());
        for (size_t n = B.bstart[b]; n < B.bstart[b + 1]; ++n) {
            const Triplet& t = B.work[n];
            S.work.push_back(t);
            S.distinct_u += 1.0 + (t.i != t.j) + (t.j != t.k);
        }
        S.bstart.push_back(S.work.size());
        for (int g = B.jstart[b]; g < B.jstart[b + 1]; ++g) S.jobs.push_back(B.jobs[g]);
    }
    S.jstart.push_back((int)S.jobs.size());
    B = S;
}

// ------------------------------------------------------------------------------------------------ slice cache
// Streamed / RI runs keep only `nslots` of the o slices X_r (with XT_r) on the device.  The whole launch order is
// known, so the cache is planned on the host: batch by batch, a slice that is missing replaces the cached slice whose
// next use lies farthest ahead (Belady), never one the batch itself needs and -- when loads are prefetched while the
// previous batch still computes (protect_prev) -- never one that batch needs.  Writes every job's slots (xr, xq) and
// the load list.  Returns false if nslots is too small.
inline bool build_slices(int o, int nslots, bool protect_prev, BatchPlan& B) {
    const size_t nbatch = B.bstart.size() - 1;
    std::vector<std::vector<int>> need(nbatch), uses(o);
    for (size_t b = 0; b < nbatch; ++b) {
        std::vector<int>& nd = need[b];
        for (int g = B.jstart[b]; g < B.jstart[b + 1]; ++g) { nd.push_back(B.jobs[g].q); nd.push_back(B.jobs[g].r); }
        std::sort(nd.begin(), nd.end());
        nd.erase(std::unique(nd.begin(), nd.end()), nd.end());
        for (int r : nd) uses[r].push_back((int)b);
    }
    std::vector<int> slot_of(o, -1), slice_in(nslots, -1);
    std::vector<size_t> nextp(o, 0);       // uses[r][nextp[r]] = first use of r in a batch after the current one
    auto has = [](const std::vector<int>& sorted, int x) { return std::binary_search(sorted.begin(), sorted.end(), x); };
    B.loads.clear();
    B.lstart.assign(1, 0);
    for (size_t b = 0; b < nbatch; ++b) {
        for (int r : need[b]) {
            if (slot_of[r] >= 0) continue;
            int best = -1;
            long long bestnext = -1;
            for (int s = 0; s < nslots; ++s) {
                const int rr = slice_in[s];
                if (rr < 0) { best = s; break; }
                if (has(need[b], rr)) continue;
                if (protect_prev && b > 0 && has(need[b - 1], rr)) continue;
                size_t& np = nextp[rr];
                while (np < uses[rr].size() && uses[rr][np] <= (int)b) ++np;
                const long long nxt = np < uses[rr].size() ? uses[rr][np] : (1LL << 40);
                if (nxt > bestnext) { bestnext = nxt; best = s; }
            }
            if (best < 0) return false;
            if (slice_in[best] >= 0) slot_of[slice_in[best]] = -1;
            slice_in[best] = r;
            slot_of[r] = best;
            B.loads.push_back({r, best});
        }
        B.lstart.push_back((int)B.loads.size());
        for (int g = B.jstart[b]; g < B.jstart[b + 1]; ++g) {
            B.jobs[g].xr = slot_of[B.jobs[g].r];
            B.jobs[g].xq = slot_of[B.jobs[g].q];
        }
    }
    return true;
}

}  // namespace tb
