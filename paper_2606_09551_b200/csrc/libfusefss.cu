// libfusefss.cu -- C ABI entry points (include/fusefss.h) and kernel launchers.  sm_100a only.
#include <cuda_runtime.h>

#include <atomic>
#include <cstdio>
#include <cstdlib>
#include <algorithm>
#include <map>
#include <mutex>
#include <string>
#include <utility>
#include <vector>

#include "program.h"
#include "aes.cuh"
#include "eval.cuh"
#include "eval_sp.cuh"
#include "eval_sp_split.cuh"
#include "keygen.cuh"
#include "post.cuh"
#include "blocks.cuh"
#include "bitslice.cuh"

namespace fsk {
namespace {

thread_local char g_cuda_err[256] = "";
thread_local cudaError_t g_cuda_code = cudaSuccess;   // code behind g_cuda_err (launch_accumulating asks for one specific failure)
std::atomic<uint64_t> g_launches{0};
thread_local int g_sms = 148;                 // SM count of the calling thread's current device (set by init_device)
std::atomic<int> g_force_g{0};                // fusefss_debug_set("force_g", v): v >= 1 forces the tree-group count (tests)
std::atomic<int> g_eval_threads{kEvalThreads};// fusefss_debug_set("eval_threads", v): CTA size of the large eval launches
std::atomic<int> g_sp_np{0};                  // fusefss_debug_set("sp_np", v): points walked in lock-step by k_eval_sp (0 = automatic)
std::atomic<int> g_sp_split{1};                // fusefss_debug_set("sp_split", v): 0 = never the lane-split kernel, 1 = for tiny launches (default), 2 = for every small launch
std::atomic<int> g_small_regs{1};             // fusefss_debug_set("small_kernels", 0): never pick the 256-thread instantiations
std::atomic<int> g_coop{1};                   // fusefss_debug_set("coop", 0): G > 1 launches take the memset + plain-launch path (tests the fallback)
const HostAes &host_aes() { static HostAes h; return h; }

int cuda_fail(cudaError_t e, const char *what) {
    std::snprintf(g_cuda_err, sizeof g_cuda_err, "%s: %s", what, cudaGetErrorString(e));
    g_cuda_code = e;
    return FUSEFSS_E_CUDA;
}
#define CU(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return cuda_fail(e_, #call); } while (0)

template <typename K> int allow_smem(K kernel, size_t bytes) {
    CU(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
    return 0;
}

// Per DEVICE, once: the PRG round keys and T0 go to that device's constant memory (__constant__ symbols are per device), and its
// SM count is recorded.  Every entry point calls this first; it also refreshes the thread-local g_sms for the current device.
struct DeviceState { bool ready = false; int sms = 0; };
int init_device() {
    static std::mutex mu;
    static std::map<int, DeviceState> devs;
    int dev = 0;
    CU(cudaGetDevice(&dev));
    std::lock_guard<std::mutex> lock(mu);
    DeviceState &D = devs[dev];
    if (!D.ready) {
        const HostAes &h = host_aes();
        uint32_t rk[kNumPrgKeys][44];
        for (int i = 0; i < kNumPrgKeys; ++i) {
            uint8_t key[16];
            for (int j = 0; j < 16; ++j) key[j] = (uint8_t)j;
            key[0] = (uint8_t)i;
            h.expand(key, rk[i]);
        }
        // prg_blocks<.., SHARED> relies on the PRG keys agreeing outside byte 0 of round key 0
        for (int i = 1; i < kNumPrgKeys; ++i)
            if ((rk[i][0] ^ rk[0][0]) & ~0xffu || rk[i][1] != rk[0][1] || rk[i][2] != rk[0][2] || rk[i][3] != rk[0][3]) return FUSEFSS_E_SPEC;
        CU(cudaMemcpyToSymbol(c_T0, h.T0, sizeof h.T0));
        CU(cudaMemcpyToSymbol(c_rk, rk, sizeof rk));
        CU(cudaDeviceGetAttribute(&D.sms, cudaDevAttrMultiProcessorCount, dev));
        D.ready = true;
    }
    g_sms = D.sms;
    return 0;
}

// Number of tree groups G in [1, gmax] for `units` (party, tile) pairs with `ntrees` trees each on `warps` persistent warps.
// A warp takes every warps-th item, so the slowest warp walks ceil(units G / warps) items of ceil(ntrees / G) trees: minimise
// that product (the launch's critical path in tree walks) and take the smallest G within 3 % of the minimum (fewer atomics).
int pick_groups(size_t units, int ntrees, int warps) {
    if (ntrees < 1) return 1;
    if (const int f = g_force_g.load()) return f < ntrees ? f : ntrees;
    auto cost = [&](int G) {
        const size_t per_warp = (units * (size_t)G + (size_t)warps - 1) / (size_t)warps;
        return per_warp * (size_t)((ntrees + G - 1) / G);
    };
    size_t best = ~(size_t)0;
    for (int G = 1; G <= ntrees; ++G) best = cost(G) < best ? cost(G) : best;
    for (int G = 1; G <= ntrees; ++G) if ((double)cost(G) <= 1.03 * (double)best) return G;
    return 1;
}

// CTA size for `warp_items` warp-sized work items: small launches use small CTAs so that the warps spread over all
// SMs (the AES kernels are bound by the per-SM shared-memory pipe), large ones use max_threads per CTA.
int threads_for(size_t warp_items, int max_threads, int min_threads = 64) {
    size_t per_sm = (warp_items + (size_t)g_sms - 1) / (size_t)g_sms;
    size_t t = per_sm * 32;
    if (t < (size_t)min_threads) t = (size_t)min_threads;
    if (t > (size_t)max_threads) t = (size_t)max_threads;
    return (int)t;
}

int grid_for(size_t warp_items, int threads) {
    size_t blocks = (warp_items + (threads / 32) - 1) / (threads / 32);
    if (blocks > (size_t)g_sms) blocks = (size_t)g_sms;
    return blocks ? (int)blocks : 1;
}

// the small per-program tables (post program, alpha, payload table, variant-1 tables) on the CURRENT device; uploaded on first use
int ensure_blob(const Program &P, const uint8_t **out) {
    int dev = 0;
    CU(cudaGetDevice(&dev));
    std::lock_guard<std::mutex> lock(P.blob_mu);
    auto it = P.dev_blobs.find(dev);
    if (it != P.dev_blobs.end()) { *out = (const uint8_t *)it->second; return 0; }
    void *d = nullptr;
    CU(cudaMalloc(&d, P.dev_blob_bytes));
    std::vector<uint8_t> h(P.dev_blob_bytes, 0);
    if (!P.ins.empty()) std::memcpy(h.data() + P.dev_ins_off, P.ins.data(), P.ins.size() * sizeof(Ins));
    if (!P.alpha.empty()) std::memcpy(h.data() + P.dev_alpha_off, P.alpha.data(), P.alpha.size() * 8);
    if (!P.payload.empty()) std::memcpy(h.data() + P.dev_payload_off, P.payload.data(), P.payload.size() * 8);
    if (!P.sp.points.empty()) std::memcpy(h.data() + P.dev_sp_points_off, P.sp.points.data(), P.sp.points.size() * sizeof(SpPoint));
    if (!P.sp.weights.empty()) std::memcpy(h.data() + P.dev_sp_weights_off, P.sp.weights.data(), P.sp.weights.size() * 8);
    if (!P.sp.delta_tab.empty()) std::memcpy(h.data() + P.dev_sp_delta_off, P.sp.delta_tab.data(), P.sp.delta_tab.size() * 8);
    if (!P.sp.clusters.empty()) std::memcpy(h.data() + P.dev_sp_clusters_off, P.sp.clusters.data(), P.sp.clusters.size() * sizeof(SpCluster));
    if (!P.sp.dense_t.empty()) std::memcpy(h.data() + P.dev_dense_t_off, P.sp.dense_t.data(), P.sp.dense_t.size() * 8);
    if (!P.sp.dense_d.empty()) std::memcpy(h.data() + P.dev_dense_d_off, P.sp.dense_d.data(), P.sp.dense_d.size() * 8);
    cudaError_t e = cudaMemcpy(d, h.data(), P.dev_blob_bytes, cudaMemcpyHostToDevice);
    if (e != cudaSuccess) { cudaFree(d); return cuda_fail(e, "cudaMemcpy(program tables)"); }
    P.dev_blobs[dev] = d;
    *out = (const uint8_t *)d;
    return 0;
}

RoundKeys seed_round_keys(uint64_t seed) {
    uint8_t key[16];
    const uint64_t inv = ~seed;
    for (int i = 0; i < 8; ++i) { key[i] = (uint8_t)(seed >> (8 * i)); key[8 + i] = (uint8_t)(inv >> (8 * i)); }
    RoundKeys rk;
    host_aes().expand(key, rk.w);
    return rk;
}

template <typename K, typename A> int launch(K kernel, int grid, int block, size_t smem, cudaStream_t st, const A &args, bool cooperative = false) {
    if (smem > 48 * 1024) {                       // opt in to > 48 KB of dynamic shared memory once per kernel (and device)
        static std::mutex mu;
        static std::vector<std::pair<const void *, int>> done;
        int dev = 0;
        CU(cudaGetDevice(&dev));
        std::lock_guard<std::mutex> lock(mu);
        const std::pair<const void *, int> id{reinterpret_cast<const void *>(kernel), dev};
        if (std::find(done.begin(), done.end(), id) == done.end()) {
            int rc = allow_smem(kernel, smem); if (rc) return rc;
            done.push_back(id);
        }
    }
    if (cooperative) {                            // the kernel uses one grid-wide barrier: all CTAs must be co-resident (grid <= #SMs)
        void *params[] = {const_cast<A *>(&args)};
        CU(cudaLaunchCooperativeKernel(reinterpret_cast<const void *>(kernel), dim3(grid), dim3(block), params, smem, st));
    } else {
        kernel<<<grid, block, smem, st>>>(args);
    }
    g_launches.fetch_add(1, std::memory_order_relaxed);
    CU(cudaGetLastError());
    return 0;
}

// Launches whose outputs are accumulated with atomics by G > 1 groups (a.zero_first): the kernel zeroes them itself behind ONE grid-wide
// barrier, which needs a cooperative launch with every CTA co-resident (grid <= #SMs, one 192-KB CTA per SM).  A context that cannot
// hold the grid -- an MPS client with an active-thread percentage, a green context or another SM partition, a co-running kernel that
// pins shared memory -- refuses it with cudaErrorCooperativeLaunchTooLarge.  Then (and with the "coop" knob off): clear the
// accumulators with cudaMemsetAsync on the same stream and launch the same kernel normally with zero_first = 0.  One more launch-sized
// memset, same results bit for bit.
template <typename K, typename A, typename Z>
int launch_accumulating(K kernel, int grid, int block, size_t smem, cudaStream_t st, A a, Z clear_accumulators) {
    if (!a.zero_first) return launch(kernel, grid, block, smem, st, a, false);
    if (g_coop.load()) {
        const int rc = launch(kernel, grid, block, smem, st, a, true);
        if (rc == 0 || g_cuda_code != cudaErrorCooperativeLaunchTooLarge) return rc;
        (void)cudaGetLastError();                  // the refusal is not sticky; clear it and take the other road
    }
    const int rc = clear_accumulators();
    if (rc) return rc;
    a.zero_first = 0;
    return launch(kernel, grid, block, smem, st, a, false);
}

// ---- dispatch on P ---------------------------------------------------------------------------------
int launch_gen_vec_p(int p, int grid, int block, cudaStream_t st, const GenVecArgs &a) {
    const size_t sm = kAesSmemBytes;
    switch (p) {
    case 1: return launch(k_gen_vec<1>, grid, block, sm, st, a);
    case 2: return launch(k_gen_vec<2>, grid, block, sm, st, a);
    case 3: return launch(k_gen_vec<3>, grid, block, sm, st, a);
    case 4: return launch(k_gen_vec<4>, grid, block, sm, st, a);
    case 5: return launch(k_gen_vec<5>, grid, block, sm, st, a);
    case 6: return launch(k_gen_vec<6>, grid, block, sm, st, a);
    case 7: return launch(k_gen_vec<7>, grid, block, sm, st, a);
    case 8: return launch(k_gen_vec<8>, grid, block, sm, st, a);
    }
    return FUSEFSS_E_SPEC;
}

// Tiny dealer launches (one warp per (32-element tile, tree) would leave at most 2 warps per SM: relu16, and the single tree per element
// of recip / rsqrt in the single-key construction): the quad-lane kernel -- four lanes per element, one child each -- cuts the per-level
// chain of a tree 4x (keygen.cuh): rsqrt v1 198 -> 72 us, relu16 v1 59 -> 27 us.  With more warps than that the SM's issue slots and lookup
// pipe are shared anyway and the quads' shuffles and replicated setup cost more than they save (recip v0: 286 -> 426 us), so those
// launches stay on k_gen_vec.
std::atomic<int> g_gen_quad{1};               // fusefss_debug_set("gen_quad", 0): always the lane-per-element dealer kernel
int launch_gen_vec(int p, size_t count, int trees, cudaStream_t st, const GenVecArgs &a) {
    const size_t tiles = (count + 31) / 32, items = tiles * (size_t)trees;
    if (g_gen_quad.load() && items <= (size_t)g_sms * 2) {
        const size_t qitems = ((count + 7) / 8) * (size_t)trees;
        const int th = threads_for(qitems, kGenThreads), grid = grid_for(qitems, th);
        switch (p) {
#define FSK_GQ_CASE(PP) case PP: return launch(k_gen_vec_quad<PP>, grid, th, kAesSmemBytes, st, a);
        FSK_GQ_CASE(1) FSK_GQ_CASE(2) FSK_GQ_CASE(3) FSK_GQ_CASE(4) FSK_GQ_CASE(5) FSK_GQ_CASE(6) FSK_GQ_CASE(7) FSK_GQ_CASE(8)
#undef FSK_GQ_CASE
        }
        return FUSEFSS_E_SPEC;
    }
    const int th = threads_for(items, kGenThreads);
    return launch_gen_vec_p(p, grid_for(items, th), th, st, a);
}

// A launch is "small" when even with every tree of every element on its own warp it leaves at most 8 warps per SM: then the
// 256-thread instantiation (255 registers per thread instead of 64) is used -- such launches live on the instruction-level
// parallelism inside a warp, not on occupancy.
bool small_launch(size_t warp_items) { return g_small_regs.load() && warp_items <= (size_t)g_sms * (kEvalThreadsSmall / 32); }

// Protocol-3 construction: ONE kernel serves eval_cmp, eval_lut, the fused call and the both-parties call.
// party = 0 / 1: that party only (slot 0); party = 2: both parties in one launch (slot b = party b).
int launch_eval_p3(const Program &P, int party, const void *const key[2], const uint64_t *xhat, size_t count,
                   uint64_t *const bits[2], uint64_t *const coeff[2], cudaStream_t st) {
    Layout L; compute_layout(P, count, &L);
    EvalArgs a{};
    a.n_slots = party == 2 ? 2 : 1; a.party0 = party == 2 ? 0 : party; a.xhat = xhat;
    for (int sl = 0; sl < a.n_slots; ++sl) { a.key[sl] = (const uint8_t *)key[sl]; a.bits_out[sl] = P.T > 0 ? bits[sl] : nullptr; a.coeff_out[sl] = P.has_lut ? coeff[sl] : nullptr; }
    a.count = count; a.s16 = L.s16; a.s8 = L.s8; a.lut_c = L.lut_c; a.vt_first = L.vt_first; a.vt_stride = L.vt_stride;
    a.lvl_stride = L.lvl_stride; a.vt_lvl_rel = L.vt_lvl_rel; a.vt_fin_rel = L.vt_fin_rel;
    a.mask = P.mask; a.n = (int)P.n; a.M = P.has_lut ? P.M : 1; a.T = P.T; a.et = (int)P.et;
    for (int t = 0; t < P.T; ++t) a.atom[t] = CmpAtomDev{P.atoms[t].c, L.bt_root[t], L.bt_cw[t], L.bt_vb[t], P.atoms[t].k, 0};
    const bool want_cmp = P.T > 0 && (a.bits_out[0] || a.bits_out[1]), want_lut = P.has_lut && (a.coeff_out[0] || a.coeff_out[1]);
    const size_t tiles = (count + 31) / 32, units = tiles * (size_t)a.n_slots;
    const size_t max_items = units * (size_t)((want_cmp ? P.T : 0) + (want_lut ? P.M - 1 : 0));
    const bool small = small_launch(max_items);
    const int cap = small ? kEvalThreadsSmall : (g_eval_threads.load() < p3_threads_for(P.p) ? g_eval_threads.load() : p3_threads_for(P.p));
    if (small) {                                   // every tree on its own warp: the chain of one tree is the critical path
        a.Gc = want_cmp ? P.T : 1; a.Gl = want_lut ? P.M - 1 : 1;
        if (const int f = g_force_g.load()) { a.Gc = f < a.Gc ? f : a.Gc; a.Gl = f < a.Gl ? f : a.Gl; }
    } else {
        a.Gc = want_cmp ? pick_groups(units, P.T, g_sms * (cap / 32)) : 1;
        a.Gl = want_lut ? pick_groups(units, P.M - 1, g_sms * (cap / 32)) : 1;
    }
    const size_t items = units * (size_t)((want_cmp ? a.Gc : 0) + (want_lut ? a.Gl : 0));
    a.zero_first = (want_cmp && a.Gc > 1) || (want_lut && a.Gl > 1);
    const int threads = small ? kEvalThreadsSmall : threads_for(items, cap);
    const int grid = small ? (int)(items < (size_t)g_sms ? items : (size_t)g_sms) : grid_for(items, threads);   // small: spread the warps over ALL SMs
    const size_t sm = kAesSmemBytes;
    auto clear = [&]() -> int {                    // what zero_outputs_and_sync would have zeroed
        for (int sl = 0; sl < a.n_slots; ++sl) {
            if (a.Gc > 1 && a.bits_out[sl]) CU(cudaMemsetAsync(a.bits_out[sl], 0, count * 8, st));
            if (a.Gl > 1 && a.coeff_out[sl]) CU(cudaMemsetAsync(a.coeff_out[sl], 0, count * 8 * (size_t)P.p, st));
        }
        return 0;
    };
#define FSK_P3_CASE(PP) case PP: return small ? launch_accumulating(k_eval_p3<PP, kEvalThreadsSmall>, grid, threads, sm, st, a, clear) \
                                              : launch_accumulating(k_eval_p3<PP, p3_threads_for(PP)>, grid, threads, sm, st, a, clear);
    switch (P.p) { FSK_P3_CASE(1) FSK_P3_CASE(2) FSK_P3_CASE(3) FSK_P3_CASE(4) FSK_P3_CASE(5) FSK_P3_CASE(6) FSK_P3_CASE(7) FSK_P3_CASE(8) }
#undef FSK_P3_CASE
    return FUSEFSS_E_SPEC;
}

// variant 1: one kernel serves eval_cmp (bits only), eval_lut (coefficients only) and the fused call (both)
// party = 0 / 1: that party only (key, bits_out, coeff_out); party = 2: both parties in ONE launch (slot b = party b)
// -- half the launches and twice the parallelism for small tensors.
int launch_eval_sp(const Program &P, int party, const void *const key[2], const uint64_t *xhat, size_t count,
                   uint64_t *const bits[2], uint64_t *const coeff[2], cudaStream_t st) {
    const uint8_t *blob = nullptr;
    int rc = ensure_blob(P, &blob); if (rc) return rc;
    Layout L; compute_layout(P, count, &L);
    EvalSpArgs a{};
    a.n_parties = party == 2 ? 2 : 1; a.party0 = party == 2 ? 0 : party; a.xhat = xhat;
    for (int sl = 0; sl < a.n_parties; ++sl) { a.key2[sl] = (const uint8_t *)key[sl]; a.bits_out2[sl] = P.T > 0 ? bits[sl] : nullptr; a.coeff_out2[sl] = P.has_lut ? coeff[sl] : nullptr; }
    a.points = (const SpPoint *)(blob + P.dev_sp_points_off); a.weights = (const uint64_t *)(blob + P.dev_sp_weights_off);
    a.delta_tab = (const uint64_t *)(blob + P.dev_sp_delta_off); a.alpha = (const uint64_t *)(blob + P.dev_alpha_off);
    a.count = count; a.s16 = L.s16; a.s8 = L.s8; a.lvl_stride = L.lvl_stride; a.vt_first = L.vt_first;
    a.vt_lvl_rel = L.vt_lvl_rel; a.vt_fin_rel = L.vt_fin_rel; a.mask = P.mask;
    a.n = (int)P.n; a.m = (int)P.m; a.p = P.p; a.T = P.T; a.n_w = P.sp.n_w; a.et = (int)P.et;
    a.n_clusters = (int)P.sp.clusters.size();
    a.cluster = (const SpCluster *)(blob + P.dev_sp_clusters_off);
    for (int w = 0; w < P.sp.n_w; ++w) { a.width[w] = P.sp.width[w]; a.bt_root[w] = L.bt_root[w]; a.bt_cw[w] = L.bt_cw[w]; a.bt_vb[w] = L.bt_vb[w]; }
    for (int t = 0; t < P.T; ++t) a.atom[t] = SpAtomDev{P.atoms[t].c, P.atoms[t].beta, P.atoms[t].k, P.atoms[t].is_theta};
    // small tensors: deal the points of an element to G warps so that the machine has >= ~8 warps per SM, then
    // spread the warps over the SMs
    const size_t tiles = (count + 31) / 32;
    int maxpts = 1;
    for (int w = 0; w < P.sp.n_w; ++w) if (P.sp.width[w].n_points > maxpts) maxpts = P.sp.width[w].n_points;
    // Group count for small launches, from a two-term model fitted to profiles/r2e_small_sweep.md: a group's critical path is
    // chain(G) = sum over clusters (shared prefix + ceil(points / G) tails) levels; up to one warp per SM sub-partition the warps
    // run at the lone-warp rate, beyond that they share the sub-partition's issue slot and the SM's shared-memory pipe (and every
    // extra group re-walks the shared prefixes), so time ~ chain(G) * max(1, warps / (4 #SMs)).  Smallest G at the minimum.
    auto model_groups = [&](size_t units) {
        int best_g = 1;
        double best = 0;
        for (int g = 1; g <= maxpts; ++g) {
            double chain = 0; int singles = 0;
            for (const SpCluster &cl : P.sp.clusters) {
                const int kf = (int)P.n - cl.tail_bits;
                if (cl.count > 1 && kf > 0) chain += kf + (double)((cl.count + g - 1) / g) * cl.tail_bits;
                else singles += cl.count;
            }
            chain += (double)((singles + g - 1) / g) * (double)P.n;
            for (int w = 0; w < P.sp.n_w; ++w)
                if (!P.sp.width[w].is_vec) chain += (double)((P.sp.width[w].n_points + g - 1) / g) * bit_tree_levels(P, P.sp.width[w].k);
            const double load = (double)(units * (size_t)g) / (4.0 * g_sms);
            const double cost = chain * (load > 1.0 ? load : 1.0);
            if (g == 1 || cost < best - 1e-9) { best = cost; best_g = g; }
        }
        return best_g;
    };
    const size_t units_sp = tiles * (size_t)a.n_parties;
    int G = units_sp < (size_t)g_sms * (kEvalSpThreads / 32) ? model_groups(units_sp) : 1;
    if (const int f = g_force_g.load()) G = f < maxpts ? f : maxpts;
    a.np = g_sp_np.load() ? g_sp_np.load() : FFS_SP_NP_SMALL;      // clamped in the kernel to its compiled maximum (1 for large launches)
    size_t items = tiles * (size_t)G * (size_t)a.n_parties;
    const bool small = small_launch(items);
    // TINY launches (even with every point of every element on its own warp at most one warp per SM sub-partition: a few hundred
    // elements): the lane-split kernel (eval_sp_split.cuh) -- the 1 + QK blocks of a level on the lanes of a group, 32 / L elements per
    // warp -- shortens the chain of one walk (one 32-element tile: 74 -> 57 us, variant 5: 107 -> 59 us).  Beyond that size the issue
    // slots are all taken anyway and its shuffles / shared-memory round keys cost more than they save (recip 1,536 elements: 115 ->
    // 125 us), so those launches stay on k_eval_sp (profiles/r2u_small_split.md).  sp_split = 2 forces it for every small launch (tests).
    const int split_l = ((P.sp.pk + 1) / 2 == 1) ? 2 : 4;
    const bool split = small && (g_sp_split.load() == 2 || (g_sp_split.load() == 1 && units_sp * (size_t)maxpts <= (size_t)g_sms * 4));
    if (split) {
        const size_t tiles_s = (count + (size_t)(32 / split_l) - 1) / (size_t)(32 / split_l);
        G = model_groups(tiles_s * (size_t)a.n_parties);
        if (const int f = g_force_g.load()) G = f < maxpts ? f : maxpts;
        items = tiles_s * (size_t)G * (size_t)a.n_parties;
    }
    a.G = G;
    a.zero_first = G > 1;
    const int cap_sp = g_eval_threads.load() < kEvalSpThreads ? g_eval_threads.load() : kEvalSpThreads;
    const int threads = small ? kEvalThreadsSmall : threads_for(items, cap_sp);
    const int grid = small ? (int)(items < (size_t)g_sms ? items : (size_t)g_sms) : grid_for(items, threads);   // small: spread the warps over ALL SMs
    const size_t sm = kAesSmemBytes;
    a.rpow = L.rpow;
    auto clear = [&]() -> int {                    // what zero_outputs_and_sync would have zeroed
        for (int sl = 0; sl < a.n_parties; ++sl) {
            if (a.bits_out2[sl]) CU(cudaMemsetAsync(a.bits_out2[sl], 0, count * 8, st));
            if (a.coeff_out2[sl]) CU(cudaMemsetAsync(a.coeff_out2[sl], 0, count * 8 * (size_t)P.p, st));
        }
        return 0;
    };
#define FSK_SPS_CASE(PP, KK) if (split && P.p == PP && P.sp.pk == KK) return launch_accumulating(k_eval_sp_split<PP, KK>, grid, threads, sm, st, a, clear);
#define FSK_SPS_ROW(KK) FSK_SPS_CASE(1, KK) FSK_SPS_CASE(2, KK) FSK_SPS_CASE(3, KK) FSK_SPS_CASE(4, KK) FSK_SPS_CASE(5, KK) \
                        FSK_SPS_CASE(6, KK) FSK_SPS_CASE(7, KK) FSK_SPS_CASE(8, KK)
    FSK_SPS_ROW(1) FSK_SPS_ROW(2) FSK_SPS_ROW(3)
#undef FSK_SPS_ROW
#undef FSK_SPS_CASE
#define FSK_SP_CASE(PP, KK) if (P.p == PP && P.sp.pk == KK) return small ? launch_accumulating(k_eval_sp<PP, KK, kEvalThreadsSmall>, grid, threads, sm, st, a, clear) \
                                                                         : launch_accumulating(k_eval_sp<PP, KK, kEvalSpThreads>, grid, threads, sm, st, a, clear);
#define FSK_SP_ROW(KK) FSK_SP_CASE(1, KK) FSK_SP_CASE(2, KK) FSK_SP_CASE(3, KK) FSK_SP_CASE(4, KK) FSK_SP_CASE(5, KK) \
                       FSK_SP_CASE(6, KK) FSK_SP_CASE(7, KK) FSK_SP_CASE(8, KK)
    FSK_SP_ROW(1) FSK_SP_ROW(2) FSK_SP_ROW(3)
#undef FSK_SP_ROW
#undef FSK_SP_CASE
    return FUSEFSS_E_SPEC;
}

// variant bit 4: the lookup by full-domain evaluation of the single key (the predicate bits still come from k_eval_sp's points)
int launch_eval_dense(const Program &P, int party, const void *const key[2], const uint64_t *xhat, size_t count,
                      uint64_t *const coeff[2], cudaStream_t st) {
    const uint8_t *blob = nullptr;
    int rc = ensure_blob(P, &blob); if (rc) return rc;
    Layout L; compute_layout(P, count, &L);
    EvalDenseArgs a{};
    a.n_parties = party == 2 ? 2 : 1; a.party0 = party == 2 ? 0 : party; a.xhat = xhat;
    for (int sl = 0; sl < a.n_parties; ++sl) { a.key2[sl] = (const uint8_t *)key[sl]; a.coeff_out2[sl] = coeff[sl]; }
    a.dense_t = (const uint64_t *)(blob + P.dev_dense_t_off); a.dense_d = (const uint64_t *)(blob + P.dev_dense_d_off);
    a.count = count; a.s16 = L.s16; a.s8 = L.s8; a.lvl_stride = L.lvl_stride; a.vt_first = L.vt_first;
    a.vt_lvl_rel = L.vt_lvl_rel; a.vt_fin_rel = L.vt_fin_rel; a.mask = P.mask; a.n = (int)P.n;
    const size_t items = count * (size_t)a.n_parties;
    const int grid = (int)(items < (size_t)g_sms ? items : (size_t)g_sms);
    switch (P.p) {
#define FSK_DN_CASE(PP) case PP: return launch(k_eval_dense<PP>, grid, kEvalThreadsSmall, kAesSmemBytes, st, a);
    FSK_DN_CASE(1) FSK_DN_CASE(2) FSK_DN_CASE(3) FSK_DN_CASE(4) FSK_DN_CASE(5) FSK_DN_CASE(6) FSK_DN_CASE(7) FSK_DN_CASE(8)
#undef FSK_DN_CASE
    }
    return FUSEFSS_E_SPEC;
}

// all four evaluation entry points end here
int launch_eval(const Program &P, int party, const void *k0, const void *k1, const uint64_t *xhat, size_t count,
                uint64_t *b0, uint64_t *b1, uint64_t *c0, uint64_t *c1, cudaStream_t st) {
    const void *const key[2] = {k0, k1};
    uint64_t *const bits[2] = {b0, b1};
    uint64_t *const coeff[2] = {c0, c1};
    if (P.dense && P.has_lut) {                     // bits from the point walks, coefficients from the full-domain traversal
        uint64_t *const none[2] = {nullptr, nullptr};
        const bool want_bits = P.T > 0 && (b0 || b1), want_coeff = c0 || c1;
        if (want_bits) { int rc = launch_eval_sp(P, party, key, xhat, count, bits, none, st); if (rc) return rc; }
        return want_coeff ? launch_eval_dense(P, party, key, xhat, count, coeff, st) : 0;
    }
    return P.variant ? launch_eval_sp(P, party, key, xhat, count, bits, coeff, st) : launch_eval_p3(P, party, key, xhat, count, bits, coeff, st);
}

PostKeyOff post_offsets(const Program &P, const Layout &L) {
    PostKeyOff k{};
    k.s8 = L.s8; k.rin = L.rin; k.rout = L.rout; k.ka = L.ka; k.kb = L.kb; k.beaver = L.beaver; k.andt = L.andt;
    k.b2a_bits = L.b2a_bits; k.b2a_a = L.b2a_a; k.s16 = L.s16; k.a2b_rho = L.a2b_rho; k.a2b_bits = L.a2b_bits; k.et = (int)P.et;
    for (int i = 0; i < P.GA2B; ++i) { k.a2b_root[i] = L.a2b_root[i]; k.a2b_cw[i] = L.a2b_cw[i]; k.a2b_vb[i] = L.a2b_vb[i]; }
    return k;
}

// post-processing launch geometry: one lane per element; programs with interactive A2B nodes walk comparison keys, so they run as
// persistent CTAs (one per SM) with the PRG tables in shared memory
template <typename K0, typename K1, typename A>
int launch_post(const Program &P, K0 plain, K1 with_a2b, size_t count, cudaStream_t st, const A &a) {
    const size_t blocks = (count + 255) / 256;
    if (P.GA2B == 0) return launch(plain, (int)blocks, 256, 0, st, a);
    return launch(with_a2b, (int)(blocks < (size_t)g_sms ? blocks : (size_t)g_sms), 256, kAesSmemBytes, st, a);
}

}  // namespace
}  // namespace fsk

using namespace fsk;

static const Program *prog_of(const fusefss_program *p) { return p ? &p->impl : nullptr; }

extern "C" {

int fusefss_compile(const fusefss_spec *spec, fusefss_program **out) {
    if (!spec || !out) return FUSEFSS_E_NULL;
    Program *P = nullptr;
    int rc = compile_program(spec, &P);
    *out = rc == 0 ? reinterpret_cast<fusefss_program *>(P) : nullptr;
    return rc;
}

void fusefss_destroy(fusefss_program *prog) {
    if (!prog) return;
    for (auto &kv : prog->impl.dev_blobs) cudaFree(kv.second);
    delete prog;
}

int fusefss_prepare(const fusefss_program *prog) {
    const Program *P = prog_of(prog);
    if (!P) return FUSEFSS_E_NULL;
    int rc = init_device(); if (rc) return rc;
    const uint8_t *blob = nullptr;
    return ensure_blob(*P, &blob);
}

int fusefss_shape(const fusefss_program *prog, fusefss_shape_t *out) {
    const Program *P = prog_of(prog);
    if (!P || !out) return FUSEFSS_E_NULL;
    *out = fusefss_shape_t{};
    out->T = P->T; out->M = P->M; out->p = P->p; out->M_A = P->MA; out->M_B = P->MB; out->G_mix = P->GMIX + P->GA2B;
    out->rounds = P->rounds; out->n_out_a = P->n_out_a; out->n_out_b = P->n_out_b; out->has_lut = P->has_lut;
    out->n_kb = P->n_kb;
    for (int t = 0; t < P->T; ++t) out->k[t] = P->atoms[t].k;
    return 0;
}

int fusefss_atom(const fusefss_program *prog, int t, uint64_t *out4) {
    const Program *P = prog_of(prog);
    if (!P || !out4) return FUSEFSS_E_NULL;
    if (t < 0 || t >= P->T) return FUSEFSS_E_SPEC;
    out4[0] = (uint64_t)P->atoms[t].k; out4[1] = P->atoms[t].c; out4[2] = (uint64_t)P->atoms[t].is_theta; out4[3] = P->atoms[t].beta;
    return 0;
}

size_t fusefss_key_bytes(const fusefss_program *prog, size_t count) {
    const Program *P = prog_of(prog);
    if (!P) return 0;
    Layout L; compute_layout(*P, count, &L);
    return L.total;
}

int fusefss_post_rounds(const fusefss_program *prog) { return prog ? prog->impl.rounds : FUSEFSS_E_NULL; }

size_t fusefss_post_msg_bytes(const fusefss_program *prog, size_t count, int round) {
    return prog ? post_msg_bytes(prog->impl, count, round) : 0;
}

size_t fusefss_online_bits(const fusefss_program *prog) {
    const Program *P = prog_of(prog);
    if (!P) return 0;
    size_t arrs = 0;
    for (int q = 0; q < P->rounds; ++q) arrs += (size_t)P->round_arr[q];
    return (size_t)P->n + (size_t)P->n * arrs + (size_t)2 * P->MB + (size_t)P->GMIX +
           (P->mask_output ? (size_t)P->n * P->n_out_a : 0);
}

// Algorithmic work per element, from the compiled program (DESIGN 5.3 / 9): AES blocks and T-table lookups.
// A group of B blocks expanded from one seed costs 15 + B + 144 B lookups (B > 1), a lone block 160.
int fusefss_cost(const fusefss_program *prog, fusefss_cost_t *out) {
    const Program *P = prog_of(prog);
    if (!P || !out) return FUSEFSS_E_NULL;
    auto grp = [](uint64_t B) { return B > 1 ? 15 + B + 144 * B : (uint64_t)160; };
    const uint64_t n = P->n, Q = (uint64_t)P->Q;
    fusefss_cost_t c{};
    if (!P->variant) {
        for (int t = 0; t < P->T; ++t) {
            const uint64_t k = (uint64_t)bit_tree_levels(*P, P->atoms[t].k);          // levels walked (early termination: k - 7)
            c.eval_cmp_aes += k + 1; c.eval_cmp_lookups += 160 * (k + 1);
            c.gen_cmp_aes += 4 * k + 4; c.gen_cmp_lookups += 2 * 160 + k * 2 * grp(2) + 2 * 160;
            c.eval_cmp_key_bytes += 16 * ((uint64_t)bit_tree_arrays(*P, P->atoms[t].k) + 1) + 8;
        }
        if (P->has_lut) {
            const uint64_t trees = (uint64_t)P->M - 1, p = (uint64_t)P->p;
            c.eval_lut_aes = trees * (n * (1 + Q) + Q); c.eval_lut_lookups = trees * (n * grp(1 + Q) + grp(Q));
            c.gen_lut_aes = trees * (4 * n * (1 + Q) + 2 * Q + 2); c.gen_lut_lookups = trees * (2 * 160 + n * 2 * grp(2 * (1 + Q)) + 2 * grp(Q));
            c.eval_lut_key_bytes = 8 * p + trees * (16 + n * (16 + 8 * p) + 8 * p);
        }
    } else {
        for (int w = 0; w < P->sp.n_w; ++w) {
            const SpWidth &W = P->sp.width[w];
            if (!W.is_vec) {
                const uint64_t k = (uint64_t)bit_tree_levels(*P, W.k);
                c.eval_cmp_aes += (uint64_t)W.n_points * (k + 1); c.eval_cmp_lookups += 160 * (uint64_t)W.n_points * (k + 1);
                c.gen_cmp_aes += 4 * k + 4; c.gen_cmp_lookups += 2 * 160 + k * 2 * grp(2) + 2 * 160;
                c.eval_cmp_key_bytes += 16 * ((uint64_t)bit_tree_arrays(*P, W.k) + 1) + 8;
                continue;
            }
            if (P->dense && P->has_lut) {                                       // full-domain traversal: every node expanded once
                const uint64_t N = 1ull << n;
                c.eval_lut_aes += 2 * (2 * N - 2) + N; c.eval_lut_lookups += (2 * N - 2) * grp(2) + 160 * N;
            }
            for (const SpCluster &cl : P->sp.clusters) {                       // fused walk: every point of the n-bit tree
                if (P->dense && P->has_lut) break;
                const uint64_t kf = n - (uint64_t)cl.tail_bits;
                const bool share = cl.count > 1 && kf > 0;
                // the shared prefix is counted once: the few levels re-walked where the cluster's second prefix forks
                // off (data dependent, ~2 per straddling lane) are overhead, not algorithmic work
                const uint64_t levels = share ? kf + (uint64_t)cl.count * (uint64_t)cl.tail_bits : (uint64_t)cl.count * n;
                const uint64_t qk = ((uint64_t)P->sp.pk + 1) / 2;
                c.eval_lut_aes += (1 + qk) * levels + qk * (uint64_t)cl.count; c.eval_lut_lookups += levels * grp(1 + qk) + grp(qk) * (uint64_t)cl.count;
            }
            const uint64_t qk = ((uint64_t)P->sp.pk + 1) / 2, pk = (uint64_t)P->sp.pk;
            c.gen_lut_aes += 4 * n * (1 + qk) + 2 * qk + 2; c.gen_lut_lookups += 2 * 160 + n * 2 * grp(2 * (1 + qk)) + 2 * grp(qk);
            c.eval_lut_key_bytes += 16 + n * (16 + 8 * pk) + 8 * pk;
        }
    }
    *out = c;
    return 0;
}

const char *fusefss_strerror(int code) {
    switch (code) {
    case FUSEFSS_OK: return "ok";
    case FUSEFSS_E_NULL: return "null pointer";
    case FUSEFSS_E_SPEC: return "ill-formed operator specification or compiled limit exceeded";
    case FUSEFSS_E_PARTY: return "party must be 0 or 1";
    case FUSEFSS_E_COUNT: return "count must be > 0";
    case FUSEFSS_E_ROUND: return "round out of range";
    case FUSEFSS_E_CUDA: return "CUDA error (see fusefss_last_cuda_error)";
    case FUSEFSS_E_OMITTED: return "call omitted for this gate type (T = 0 or m = 1)";
    case FUSEFSS_E_WORKSPACE: return "workspace smaller than fusefss_gate_workspace_bytes()";
    case FUSEFSS_E_DEBUG: return "unknown debug knob";
    case FUSEFSS_E_STATIC: return "post-processing program longer than FUSEFSS_NOALLOC_MAX_INS instructions: use fusefss_post_fused";
    }
    return "unknown error";
}
const char *fusefss_last_cuda_error(void) { return g_cuda_err; }
int fusefss_debug_set(const char *knob, long value) {
    if (!knob) return FUSEFSS_E_NULL;
    const std::string k(knob);
    if (k == "force_g") { g_force_g.store(value >= 1 ? (int)value : 0); return 0; }
    if (k == "eval_threads") { g_eval_threads.store(value >= 32 && value <= kEvalThreads && value % 32 == 0 ? (int)value : kEvalThreads); return 0; }
    if (k == "small_kernels") { g_small_regs.store(value ? 1 : 0); return 0; }
    if (k == "sp_np") { g_sp_np.store(value >= 1 ? (int)value : 0); return 0; }
    if (k == "gen_quad") { g_gen_quad.store(value ? 1 : 0); return 0; }
    if (k == "coop") { g_coop.store(value ? 1 : 0); return 0; }
    if (k == "sp_split") { g_sp_split.store(value >= 0 && value <= 2 ? (int)value : 1); return 0; }
    return FUSEFSS_E_DEBUG;
}
uint64_t fusefss_launch_count(void) { return g_launches.load(); }

int fusefss_keygen(const fusefss_program *prog, const uint64_t *r_in_dev, const uint64_t *r_out_dev, uint64_t seed,
                   uint64_t first_elem, size_t count, void *key0_dev, void *key1_dev, void *stream) {
    return fusefss_keygen_parts(prog, r_in_dev, r_out_dev, seed, first_elem, count, key0_dev, key1_dev,
                                FUSEFSS_GEN_CMP | FUSEFSS_GEN_LUT | FUSEFSS_GEN_SHARES, stream);
}

int fusefss_keygen_parts(const fusefss_program *prog, const uint64_t *r_in_dev, const uint64_t *r_out_dev, uint64_t seed,
                         uint64_t first_elem, size_t count, void *key0_dev, void *key1_dev, int parts, void *stream) {
    const Program *P = prog_of(prog);
    if (!P || !r_in_dev || !key0_dev || !key1_dev) return FUSEFSS_E_NULL;
    if (P->mask_output && !r_out_dev) return FUSEFSS_E_NULL;
    if (count == 0) return FUSEFSS_E_COUNT;
    int rc = init_device(); if (rc) return rc;
    const uint8_t *blob = nullptr;
    rc = ensure_blob(*P, &blob); if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    Layout L; compute_layout(*P, count, &L);
    const RoundKeys rk = seed_round_keys(seed);
    const uint64_t *alpha_dev = (const uint64_t *)(blob + P->dev_alpha_off);
    const uint64_t *payload_dev = (const uint64_t *)(blob + P->dev_payload_off);
    const size_t tiles = (count + 31) / 32;
    const size_t smem = kAesSmemBytes;
    // ---- arguments of the three dealer kernels (built unconditionally: host work only) -------------------------
    bool has_bit = false, has_vec = false;
    int vec_p = 1, vec_trees = 0;
    GenBitArgs ab{};
    ab.key0 = (uint8_t *)key0_dev; ab.key1 = (uint8_t *)key1_dev; ab.r_in = r_in_dev;
    ab.count = count; ab.s16 = L.s16; ab.first_elem = first_elem; ab.mask = P->mask; ab.rk = rk; ab.et = (int)P->et;
    GenVecArgs av{};
    av.key0 = (uint8_t *)key0_dev; av.key1 = (uint8_t *)key1_dev; av.r_in = r_in_dev; av.alpha = alpha_dev; av.payload = payload_dev;
    av.count = count; av.s16 = L.s16; av.s8 = L.s8; av.vt_first = L.vt_first; av.vt_stride = L.vt_stride; av.lvl_stride = L.lvl_stride;
    av.vt_lvl_rel = L.vt_lvl_rel; av.vt_fin_rel = L.vt_fin_rel; av.first_elem = first_elem; av.mask = P->mask;
    av.n = (int)P->n; av.m = (int)P->m; av.rk = rk;
    if (P->variant) {                                   // variant 1: one tree per view width (DESIGN 9)
        ab.T = P->sp.n_w;
        for (int w = 0; w < P->sp.n_w; ++w) {
            const bool vec = P->sp.width[w].is_vec != 0;
            has_bit = has_bit || !vec; has_vec = has_vec || vec;
            ab.atom[w] = GenAtomDev{0, 0, L.bt_root[w], L.bt_cw[w], L.bt_vb[w], vec ? 0 : P->sp.width[w].k, 0};
        }
        av.M = 2; av.sp = 1; vec_p = P->sp.pk; vec_trees = 1;
    } else {
        has_bit = P->T > 0; has_vec = P->has_lut != 0;
        ab.T = P->T;
        for (int t = 0; t < P->T; ++t)
            ab.atom[t] = GenAtomDev{P->atoms[t].c, P->atoms[t].beta, L.bt_root[t], L.bt_cw[t], L.bt_vb[t], P->atoms[t].k, P->atoms[t].is_theta};
        av.M = P->M; av.xpoly = (int)P->xpoly; av.polys = (int)P->r; av.d = (int)P->d; vec_p = P->p; vec_trees = P->M - 1;
    }
    GenMiscArgs am{};
    {
        GenMiscArgs &a = am;
        a.key0 = (uint8_t *)key0_dev; a.key1 = (uint8_t *)key1_dev; a.r_in = r_in_dev; a.r_out = r_out_dev;
        a.alpha = alpha_dev; a.payload = payload_dev;
        a.count = count; a.s8 = L.s8; a.lut_c = L.lut_c; a.rin = L.rin; a.rout = L.rout; a.ka = L.ka; a.kb = L.kb;
        a.beaver = L.beaver; a.andt = L.andt; a.b2a_bits = L.b2a_bits; a.b2a_a = L.b2a_a;
        a.first_elem = first_elem; a.mask = P->mask;
        a.n = (int)P->n; a.m = (int)P->m; a.M = P->M; a.p = P->p; a.has_lut = P->variant ? 0 : P->has_lut; a.mask_output = (int)P->mask_output;
        a.n_out_a = P->n_out_a; a.n_ka = (int)P->kappa_a.size(); a.n_kb_spec = (int)P->kappa_b.size(); a.n_carry = P->n_carry;
        a.rpow = L.rpow; a.n_rpow = (P->variant && P->xpoly) ? (int)P->d : 0;
        a.xpoly = (int)P->xpoly; a.polys = (int)P->r; a.d = (int)P->d;
        a.T = P->variant ? 0 : P->T; a.MA = P->MA; a.MB = P->MB; a.GMIX = P->GMIX; a.rk = rk;
        for (int g = 0; g < P->MA; ++g) if (P->ma_is_x[g]) a.ma_is_x |= 1ull << g;
        for (int t = 0; t < a.n_ka; ++t) { a.ka_kind[t] = P->kappa_a[t].kind; a.ka_arg[t] = P->kappa_a[t].arg; }
        for (int t = 0; t < a.n_kb_spec; ++t) { a.kb_kind[t] = P->kappa_b[t].kind; a.kb_arg[t] = P->kappa_b[t].arg; }
        for (int t = 0; t < a.T; ++t)
            a.atom[t] = GenAtomDev{P->atoms[t].c, P->atoms[t].beta, 0, 0, 0, P->atoms[t].k, P->atoms[t].is_theta};
        a.a2b_rho = L.a2b_rho; a.a2b_bits = L.a2b_bits; a.GA2B = P->GA2B;
        for (int i = 0; i < P->GA2B; ++i) a.a2b_bit[i] = P->a2b_bit[i];
    }
    const size_t bit_items = tiles * (size_t)ab.T, vec_items = tiles * (size_t)vec_trees;
    // TINY tensors, whole key at once: ONE launch for the three parts (k_gen_tiny) -- a launch costs 9-10 us of launch + table fill
    const int all_parts = FUSEFSS_GEN_CMP | FUSEFSS_GEN_LUT | FUSEFSS_GEN_SHARES;
    if (g_gen_quad.load() && (parts & all_parts) == all_parts && P->GA2B == 0 && (!has_vec || vec_items <= (size_t)g_sms * 2) &&
        (!has_bit || bit_items <= (size_t)g_sms * 8)) {
        GenTinyArgs t{};
        t.bit = ab; t.vec = av; t.misc = am; t.has_bit = has_bit ? 1 : 0; t.has_vec = has_vec ? 1 : 0;
        size_t items = tiles;
        if (has_bit && bit_items > items) items = bit_items;
        if (has_vec && ((count + 7) / 8) * (size_t)vec_trees > items) items = ((count + 7) / 8) * (size_t)vec_trees;
        const int th = threads_for(items, kGenThreads), grid = grid_for(items, th);
        switch (has_vec ? vec_p : 1) {
#define FSK_GT_CASE(PP) case PP: return launch(k_gen_tiny<PP>, grid, th, smem, st, t);
        FSK_GT_CASE(1) FSK_GT_CASE(2) FSK_GT_CASE(3) FSK_GT_CASE(4) FSK_GT_CASE(5) FSK_GT_CASE(6) FSK_GT_CASE(7) FSK_GT_CASE(8)
#undef FSK_GT_CASE
        }
        return FUSEFSS_E_SPEC;
    }
    if (has_bit && (parts & FUSEFSS_GEN_CMP)) {
        const int th = threads_for(bit_items, kGenThreads);
        rc = launch(k_gen_bit, grid_for(bit_items, th), th, smem, st, ab);
        if (rc) return rc;
    }
    if (has_vec && (parts & FUSEFSS_GEN_LUT)) {
        rc = launch_gen_vec(vec_p, count, vec_trees, st, av);
        if (rc) return rc;
    }
    if (parts & FUSEFSS_GEN_SHARES) {
        const int th = threads_for(tiles, kGenThreads), grid = grid_for(tiles, th);
        rc = launch(k_gen_misc, grid, th, kAesSmemBytes, st, am);
        if (rc) return rc;
        if (P->GA2B > 0) {                              // the A2B nodes' comparison keys f_{rho_i mod 2^j, 1} (DESIGN 15): part of the shares section
            GenBitArgs ab{};
            ab.key0 = (uint8_t *)key0_dev; ab.key1 = (uint8_t *)key1_dev; ab.r_in = r_in_dev;
            ab.count = count; ab.s16 = L.s16; ab.first_elem = first_elem; ab.mask = P->mask; ab.T = P->GA2B; ab.rk = rk; ab.et = (int)P->et;
            ab.slot_t0 = 0x400;
            for (int i = 0; i < P->GA2B; ++i) ab.atom[i] = GenAtomDev{0, 0, L.a2b_root[i], L.a2b_cw[i], L.a2b_vb[i], P->a2b_bit[i], 2};
            const int th2 = threads_for(tiles * P->GA2B, kGenThreads);
            rc = launch(k_gen_bit, grid_for(tiles * P->GA2B, th2), th2, kAesSmemBytes, st, ab);
            if (rc) return rc;
        }
    }
    return 0;
}

int fusefss_eval_cmp(int party, const fusefss_program *prog, const void *key_dev, const uint64_t *xhat_dev, size_t count,
                     uint64_t *bits_out_dev, void *stream) {
    const Program *P = prog_of(prog);
    if (!P || !key_dev || !xhat_dev || !bits_out_dev) return FUSEFSS_E_NULL;
    if (party != 0 && party != 1) return FUSEFSS_E_PARTY;
    if (count == 0) return FUSEFSS_E_COUNT;
    if (P->T == 0) return FUSEFSS_E_OMITTED;
    int rc = init_device(); if (rc) return rc;
    return launch_eval(*P, party, key_dev, nullptr, xhat_dev, count, bits_out_dev, nullptr, nullptr, nullptr, (cudaStream_t)stream);
}

int fusefss_eval_lut(int party, const fusefss_program *prog, const void *key_dev, const uint64_t *xhat_dev, size_t count,
                     uint64_t *coeff_out_dev, void *stream) {
    const Program *P = prog_of(prog);
    if (!P || !key_dev || !xhat_dev || !coeff_out_dev) return FUSEFSS_E_NULL;
    if (party != 0 && party != 1) return FUSEFSS_E_PARTY;
    if (count == 0) return FUSEFSS_E_COUNT;
    if (!P->has_lut) return FUSEFSS_E_OMITTED;
    int rc = init_device(); if (rc) return rc;
    return launch_eval(*P, party, key_dev, nullptr, xhat_dev, count, nullptr, nullptr, coeff_out_dev, nullptr, (cudaStream_t)stream);
}

int fusefss_eval_fused(int party, const fusefss_program *prog, const void *key_dev, const uint64_t *xhat_dev, size_t count,
                       uint64_t *bits_out_dev, uint64_t *coeff_out_dev, void *stream) {
    const Program *P = prog_of(prog);
    if (!P || !key_dev || !xhat_dev) return FUSEFSS_E_NULL;
    if ((P->T > 0 && !bits_out_dev) || (P->has_lut && !coeff_out_dev)) return FUSEFSS_E_NULL;
    if (party != 0 && party != 1) return FUSEFSS_E_PARTY;
    if (count == 0) return FUSEFSS_E_COUNT;
    if (P->T == 0 && !P->has_lut) return FUSEFSS_E_OMITTED;
    int rc = init_device(); if (rc) return rc;
    return launch_eval(*P, party, key_dev, nullptr, xhat_dev, count, bits_out_dev, nullptr, coeff_out_dev, nullptr, (cudaStream_t)stream);
}

int fusefss_eval_fused_both(const fusefss_program *prog, const void *key0_dev, const void *key1_dev, const uint64_t *xhat_dev,
                            size_t count, uint64_t *bits0_dev, uint64_t *bits1_dev, uint64_t *coeff0_dev, uint64_t *coeff1_dev,
                            void *stream) {
    const Program *P = prog_of(prog);
    if (!P || !key0_dev || !key1_dev || !xhat_dev) return FUSEFSS_E_NULL;
    if ((P->T > 0 && (!bits0_dev || !bits1_dev)) || (P->has_lut && (!coeff0_dev || !coeff1_dev))) return FUSEFSS_E_NULL;
    if (count == 0) return FUSEFSS_E_COUNT;
    if (P->T == 0 && !P->has_lut) return FUSEFSS_E_OMITTED;
    int rc = init_device(); if (rc) return rc;
    return launch_eval(*P, 2, key0_dev, key1_dev, xhat_dev, count, bits0_dev, bits1_dev, coeff0_dev, coeff1_dev, (cudaStream_t)stream);
}

int fusefss_post(int party, const fusefss_program *prog, const void *key_dev, const uint64_t *xhat_dev,
                 const uint64_t *bits_dev, const uint64_t *coeff_dev, size_t count, int round, const void *msg_in_dev,
                 void *msg_out_dev, uint64_t *y_out_dev, uint64_t *z_out_dev, void *stream) {
    const Program *P = prog_of(prog);
    if (!P || !key_dev || !xhat_dev) return FUSEFSS_E_NULL;
    if (party != 0 && party != 1) return FUSEFSS_E_PARTY;
    if (count == 0) return FUSEFSS_E_COUNT;
    if (round < 0 || round > P->rounds) return FUSEFSS_E_ROUND;
    if ((P->T > 0 && !bits_dev) || (P->has_lut && !coeff_dev)) return FUSEFSS_E_NULL;
    if (round < P->rounds && !msg_out_dev) return FUSEFSS_E_NULL;
    if (round > 0 && !msg_in_dev) return FUSEFSS_E_NULL;
    if (round == P->rounds && ((P->n_out_a > 0 && !y_out_dev) || (P->n_out_b > 0 && !z_out_dev))) return FUSEFSS_E_NULL;
    int rc = init_device(); if (rc) return rc;
    const uint8_t *blob = nullptr;
    rc = ensure_blob(*P, &blob); if (rc) return rc;
    Layout L; compute_layout(*P, count, &L);
    PostArgs a{};
    a.ins = (const Ins *)(blob + P->dev_ins_off); a.n_ins = (int)P->ins.size();
    a.party = party; a.round = round; a.rounds = P->rounds; a.mask_output = (int)P->mask_output;
    a.n_out_a = P->n_out_a; a.n_out_b = P->n_out_b;
    a.key = (const uint8_t *)key_dev; a.xhat = xhat_dev; a.bits = bits_dev; a.coeff = coeff_dev;
    a.msg_in = (const uint8_t *)msg_in_dev; a.msg_out = (uint8_t *)msg_out_dev; a.y_out = y_out_dev; a.z_out = z_out_dev;
    a.count = count; a.mask = P->mask; a.k = post_offsets(*P, L);
    a.round_off[0] = 0;
    for (int q = 0; q < kMaxRounds; ++q) {
        a.round_off[q + 1] = a.round_off[q] + post_msg_bytes(*P, count, q);
        a.round_arr[q] = P->round_arr[q]; a.round_bits[q] = P->round_bits[q];
    }
    return launch_post(*P, k_post_round<false>, k_post_round<true>, count, (cudaStream_t)stream, a);
}

int fusefss_post_fused(const fusefss_program *prog, const void *key0_dev, const void *key1_dev, const uint64_t *xhat_dev,
                       const uint64_t *bits0_dev, const uint64_t *bits1_dev, const uint64_t *coeff0_dev,
                       const uint64_t *coeff1_dev, size_t count, uint64_t *y0_dev, uint64_t *y1_dev, uint64_t *z0_dev,
                       uint64_t *z1_dev, void *stream) {
    const Program *P = prog_of(prog);
    if (!P || !key0_dev || !key1_dev || !xhat_dev) return FUSEFSS_E_NULL;
    if (count == 0) return FUSEFSS_E_COUNT;
    if ((P->T > 0 && (!bits0_dev || !bits1_dev)) || (P->has_lut && (!coeff0_dev || !coeff1_dev))) return FUSEFSS_E_NULL;
    if ((P->n_out_a > 0 && (!y0_dev || !y1_dev)) || (P->n_out_b > 0 && (!z0_dev || !z1_dev))) return FUSEFSS_E_NULL;
    int rc = init_device(); if (rc) return rc;
    const uint8_t *blob = nullptr;
    rc = ensure_blob(*P, &blob); if (rc) return rc;
    Layout L; compute_layout(*P, count, &L);
    PostFusedArgs a{};
    a.ins = (const Ins *)(blob + P->dev_ins_off); a.n_ins = (int)P->ins.size();
    a.mask_output = (int)P->mask_output; a.n_out_a = P->n_out_a; a.n_out_b = P->n_out_b;
    a.key[0] = (const uint8_t *)key0_dev; a.key[1] = (const uint8_t *)key1_dev; a.xhat = xhat_dev;
    a.bits[0] = bits0_dev; a.bits[1] = bits1_dev; a.coeff[0] = coeff0_dev; a.coeff[1] = coeff1_dev;
    a.y_out[0] = y0_dev; a.y_out[1] = y1_dev; a.z_out[0] = z0_dev; a.z_out[1] = z1_dev;
    a.count = count; a.mask = P->mask; a.k = post_offsets(*P, L);
    return launch_post(*P, k_post_fused<false>, k_post_fused<true>, count, (cudaStream_t)stream, a);
}

// ---- vector-block glue (App. G) -------------------------------------------
int fusefss_share_open(const fusefss_program *prog, const void *key0_dev, const void *key1_dev, const uint64_t *x0_dev,
                       const uint64_t *x1_dev, size_t count, uint64_t public_offset, uint64_t *xhat_out_dev, void *stream) {
    const Program *P = prog_of(prog);
    if (!P || !key0_dev || !key1_dev || !x0_dev || !x1_dev || !xhat_out_dev) return FUSEFSS_E_NULL;
    if (count == 0) return FUSEFSS_E_COUNT;
    Layout L; compute_layout(*P, count, &L);
    OpenArgs a{x0_dev, x1_dev, (const uint8_t *)key0_dev, (const uint8_t *)key1_dev, L.rin, count, P->mask, public_offset & P->mask, xhat_out_dev};
    return launch(k_share_open, (int)((count + 255) / 256), 256, 0, (cudaStream_t)stream, a);
}

int fusefss_open_output(uint32_t n_bits, const uint64_t *y0_dev, const uint64_t *y1_dev, size_t count, uint64_t public_offset,
                        uint64_t *yhat_out_dev, void *stream) {
    if (!y0_dev || !y1_dev || !yhat_out_dev) return FUSEFSS_E_NULL;
    if (count == 0) return FUSEFSS_E_COUNT;
    if (n_bits < 1 || n_bits > 64) return FUSEFSS_E_SPEC;
    const uint64_t mask = n_bits >= 64 ? ~0ull : ((1ull << n_bits) - 1ull);
    OpenOutArgs a{y0_dev, y1_dev, count, mask, public_offset & mask, yhat_out_dev};
    return launch(k_open_output, (int)((count + 255) / 256), 256, 0, (cudaStream_t)stream, a);
}

int fusefss_row_sum(uint32_t n_bits, const uint64_t *in_dev, size_t rows, size_t cols, uint64_t *out_dev, void *stream) {
    if (!in_dev || !out_dev) return FUSEFSS_E_NULL;
    if (rows == 0 || cols == 0) return FUSEFSS_E_COUNT;
    if (n_bits < 1 || n_bits > 64) return FUSEFSS_E_SPEC;
    RowSumArgs a{in_dev, out_dev, rows, cols, n_bits >= 64 ? ~0ull : ((1ull << n_bits) - 1ull)};
    return launch(k_row_sum, (int)((rows * 32 + 255) / 256), 256, 0, (cudaStream_t)stream, a);
}

int fusefss_sub_bcast(uint32_t n_bits, const uint64_t *x_dev, const uint64_t *mu_dev, size_t count, size_t cols, uint64_t *out_dev, void *stream) {
    if (!x_dev || !mu_dev || !out_dev) return FUSEFSS_E_NULL;
    if (count == 0 || cols == 0) return FUSEFSS_E_COUNT;
    if (n_bits < 1 || n_bits > 64) return FUSEFSS_E_SPEC;
    SubBcastArgs a{x_dev, mu_dev, out_dev, count, cols, n_bits >= 64 ? ~0ull : ((1ull << n_bits) - 1ull)};
    return launch(k_sub_bcast, (int)((count + 255) / 256), 256, 0, (cudaStream_t)stream, a);
}

size_t fusefss_mul_triple_bytes(size_t count) { return 3 * ((count * 8 + 255) & ~(size_t)255); }

int fusefss_mul_keygen(uint32_t n_bits, uint64_t seed, uint64_t first_elem, size_t count, void *t0_dev, void *t1_dev, void *stream) {
    if (!t0_dev || !t1_dev) return FUSEFSS_E_NULL;
    if (count == 0) return FUSEFSS_E_COUNT;
    if (n_bits < 1 || n_bits > 64) return FUSEFSS_E_SPEC;
    int rc = init_device(); if (rc) return rc;
    MulGenArgs a{};
    a.t0 = (uint8_t *)t0_dev; a.t1 = (uint8_t *)t1_dev; a.count = count; a.s8 = (count * 8 + 255) & ~(size_t)255;
    a.first_elem = first_elem; a.mask = n_bits >= 64 ? ~0ull : ((1ull << n_bits) - 1ull); a.rk = seed_round_keys(seed);
    const size_t tiles = (count + 31) / 32;
    const int th = threads_for(tiles, kGenThreads);
    return launch(k_mul_gen, grid_for(tiles, th), th, kAesSmemBytes, (cudaStream_t)stream, a);
}

int fusefss_mul_fused(uint32_t n_bits, const uint64_t *x0_dev, const uint64_t *x1_dev, const uint64_t *y0_dev, const uint64_t *y1_dev,
                      const void *t0_dev, const void *t1_dev, size_t count, size_t cols, uint64_t *z0_dev, uint64_t *z1_dev, void *stream) {
    if (!x0_dev || !x1_dev || !y0_dev || !y1_dev || !t0_dev || !t1_dev || !z0_dev || !z1_dev) return FUSEFSS_E_NULL;
    if (count == 0 || cols == 0) return FUSEFSS_E_COUNT;
    if (n_bits < 1 || n_bits > 64) return FUSEFSS_E_SPEC;
    MulArgs a{x0_dev, x1_dev, y0_dev, y1_dev, (const uint8_t *)t0_dev, (const uint8_t *)t1_dev, z0_dev, z1_dev, count, cols,
              (count * 8 + 255) & ~(size_t)255, n_bits >= 64 ? ~0ull : ((1ull << n_bits) - 1ull)};
    return launch(k_mul_fused, (int)((count + 255) / 256), 256, 0, (cudaStream_t)stream, a);
}

// workspace: key0 | key1 | bits0 | bits1 | coeff0[p] | coeff1[p] | 2 x { r_in | r_out[na] | xhat | y0[na] | y1[na] | z0 | z1 }
// (the input / output arrays are double-buffered so that the copies of chunk i+1 / i-1 overlap the kernels of chunk i)
static size_t ws_io_arrays(const Program &P) { return 4 + (size_t)3 * (P.n_out_a > 0 ? P.n_out_a : 1); }
static size_t ws_u64_arrays(const Program &P) { return 2 + (size_t)2 * P.p + 2 * ws_io_arrays(P); }

size_t fusefss_gate_workspace_bytes(const fusefss_program *prog, size_t chunk) {
    const Program *P = prog_of(prog);
    if (!P || chunk == 0) return 0;
    Layout L; compute_layout(*P, chunk, &L);
    return 2 * L.total + ws_u64_arrays(*P) * L.s8;
}

namespace {
// one copy stream and a few events per device for fusefss_gate_host, created on first use and kept for the life of the process
struct HostPipe {
    cudaStream_t copy = nullptr; cudaEvent_t in_ready[2] = {}, in_free[2] = {}, out_ready[2] = {}, out_free[2] = {};
    std::mutex call_mu;                                        // the events are shared by the calls on THIS device: one call at a time per device
};
int host_pipe(HostPipe **out) {
    static std::mutex mu;
    static std::map<int, HostPipe> pipes;
    int dev = 0;
    CU(cudaGetDevice(&dev));
    std::lock_guard<std::mutex> lock(mu);
    HostPipe &hp = pipes[dev];
    if (!hp.copy) {
        cudaStream_t cs = nullptr;
        CU(cudaStreamCreateWithFlags(&cs, cudaStreamNonBlocking));
        for (int i = 0; i < 2; ++i) {
            CU(cudaEventCreateWithFlags(&hp.in_ready[i], cudaEventDisableTiming)); CU(cudaEventCreateWithFlags(&hp.in_free[i], cudaEventDisableTiming));
            CU(cudaEventCreateWithFlags(&hp.out_ready[i], cudaEventDisableTiming)); CU(cudaEventCreateWithFlags(&hp.out_free[i], cudaEventDisableTiming));
        }
        hp.copy = cs;
    }
    *out = &hp;
    return 0;
}
}  // namespace

// Chunk i: [copy stream] H2D of its inputs into buffer i % 2 -> [caller's stream] keygen, evaluation, post-processing -> [copy stream]
// D2H of its outputs.  The copies of chunks i+1 (in) and i-1 (out) run while chunk i computes; one call at a time per device.
int fusefss_gate_host(const fusefss_program *prog, const uint64_t *r_in, const uint64_t *r_out, const uint64_t *xhat,
                      uint64_t seed, size_t count, size_t chunk, void *workspace_dev, size_t workspace_bytes, uint64_t *y0,
                      uint64_t *y1, uint64_t *z0, uint64_t *z1, void *stream) {
    const Program *P = prog_of(prog);
    if (!P || !r_in || !xhat || !workspace_dev) return FUSEFSS_E_NULL;
    if (chunk && workspace_bytes < fusefss_gate_workspace_bytes(prog, chunk)) return FUSEFSS_E_WORKSPACE;
    if (P->mask_output && !r_out) return FUSEFSS_E_NULL;
    if ((P->n_out_a > 0 && (!y0 || !y1)) || (P->n_out_b > 0 && (!z0 || !z1))) return FUSEFSS_E_NULL;
    if (count == 0 || chunk == 0) return FUSEFSS_E_COUNT;
    int rc = init_device(); if (rc) return rc;
    HostPipe *hp = nullptr;
    rc = host_pipe(&hp); if (rc) return rc;
    std::lock_guard<std::mutex> call_lock(hp->call_mu);        // per device: calls on different GPUs of one process run concurrently
    cudaStream_t st = (cudaStream_t)stream, cs = hp->copy;
    Layout L; compute_layout(*P, chunk, &L);
    const int na = P->n_out_a > 0 ? P->n_out_a : 1;
    uint8_t *ws = (uint8_t *)workspace_dev;
    uint8_t *key0 = ws, *key1 = ws + L.total;
    uint8_t *q = ws + 2 * L.total;
    auto take = [&](size_t arrays) { uint64_t *r = (uint64_t *)q; q += arrays * L.s8; return r; };
    uint64_t *d_b0 = take(1), *d_b1 = take(1), *d_c0 = take(P->p), *d_c1 = take(P->p);
    struct Io { uint64_t *rin, *rout, *xhat, *y0, *y1, *z0, *z1; } io[2];
    for (int b = 0; b < 2; ++b) io[b] = Io{take(1), take(na), take(1), take(na), take(na), take(1), take(1)};
    const size_t n_chunks = (count + chunk - 1) / chunk;
    auto upload = [&](size_t i) -> int {                       // [copy stream] inputs of chunk i
        const size_t first = i * chunk, c = count - first < chunk ? count - first : chunk;
        const Io &B = io[i & 1];
        if (i >= 2) CU(cudaStreamWaitEvent(cs, hp->in_free[i & 1], 0));          // chunk i-2 has consumed this buffer
        CU(cudaMemcpyAsync(B.rin, r_in + first, c * 8, cudaMemcpyHostToDevice, cs));
        CU(cudaMemcpyAsync(B.xhat, xhat + first, c * 8, cudaMemcpyHostToDevice, cs));
        if (P->mask_output)
            for (int j = 0; j < P->n_out_a; ++j)
                CU(cudaMemcpyAsync(B.rout + (size_t)j * c, r_out + (size_t)j * count + first, c * 8, cudaMemcpyHostToDevice, cs));
        CU(cudaEventRecord(hp->in_ready[i & 1], cs));
        return 0;
    };
    auto pipeline = [&]() -> int {
    CU(cudaEventRecord(hp->out_free[0], st)); CU(cudaEventRecord(hp->out_free[1], st));
    CU(cudaStreamWaitEvent(cs, hp->out_free[0], 0));           // order the copy stream after the caller's earlier work on `stream`
    rc = upload(0); if (rc) return rc;
    if (n_chunks > 1) { rc = upload(1); if (rc) return rc; }
    for (size_t i = 0; i < n_chunks; ++i) {
        const size_t first = i * chunk, c = count - first < chunk ? count - first : chunk;
        const Io &B = io[i & 1];
        CU(cudaStreamWaitEvent(st, hp->in_ready[i & 1], 0));
        if (i >= 2) CU(cudaStreamWaitEvent(st, hp->out_free[i & 1], 0));         // chunk i-2's outputs have left this buffer
        rc = fusefss_keygen(prog, B.rin, B.rout, seed, first, c, key0, key1, st); if (rc) return rc;
        if (P->T > 0 || P->has_lut) {
            rc = fusefss_eval_fused_both(prog, key0, key1, B.xhat, c, d_b0, d_b1, d_c0, d_c1, st); if (rc) return rc;
        }
        rc = fusefss_post_fused(prog, key0, key1, B.xhat, d_b0, d_b1, d_c0, d_c1, c, B.y0, B.y1, B.z0, B.z1, st); if (rc) return rc;
        CU(cudaEventRecord(hp->in_free[i & 1], st));
        CU(cudaEventRecord(hp->out_ready[i & 1], st));
        CU(cudaStreamWaitEvent(cs, hp->out_ready[i & 1], 0));                    // [copy stream] outputs of chunk i
        for (int j = 0; j < P->n_out_a; ++j) {
            CU(cudaMemcpyAsync(y0 + (size_t)j * count + first, B.y0 + (size_t)j * c, c * 8, cudaMemcpyDeviceToHost, cs));
            CU(cudaMemcpyAsync(y1 + (size_t)j * count + first, B.y1 + (size_t)j * c, c * 8, cudaMemcpyDeviceToHost, cs));
        }
        if (P->n_out_b > 0) {
            CU(cudaMemcpyAsync(z0 + first, B.z0, c * 8, cudaMemcpyDeviceToHost, cs));
            CU(cudaMemcpyAsync(z1 + first, B.z1, c * 8, cudaMemcpyDeviceToHost, cs));
        }
        CU(cudaEventRecord(hp->out_free[i & 1], cs));
        if (i + 2 < n_chunks) { rc = upload(i + 2); if (rc) return rc; }
    }
    CU(cudaStreamSynchronize(cs));
    CU(cudaStreamSynchronize(st));
    return 0;
    };
    rc = pipeline();
    if (rc) {                                                  // a step failed mid-pipeline: copies into / out of the caller's host buffers and kernels on the
        (void)cudaStreamSynchronize(cs);                       // workspace may still be in flight.  Drain both streams before reporting, so that the caller
        (void)cudaStreamSynchronize(st);                       // may free its buffers on error (the text of the first failure stays in fusefss_last_cuda_error)
    }
    return rc;
}

}  // extern "C"

// ---- fusefss_post_fused_noalloc: the fused post-processing pass for callers that must not allocate ------------------------
// (include/fusefss.h says who they are: servers whose allocator already owns all of HBM, latency-bound online loops that cannot
// take cudaMalloc's device-wide synchronisation, processes under a fixed device-memory quota.)
//
// k_post_fused interprets the program's instruction table from global memory.  fusefss_post_fused keeps that table in a buffer it
// cudaMalloc's on first use (ensure_blob); here the table goes into an array that is part of the module image instead, so it exists
// on every GPU that loads the library, from module load to process exit: kStaticPostIns * sizeof(Ins) = 2048 * 24 B = 48 KB.
//
// One array per device, shared by all calls, programs and streams.  It keeps whatever the last call wrote; each call overwrites
// the first n_ins entries on its own stream before its kernel and the kernel reads only those, so nothing needs clearing.  Calls
// that can overlap on the GPU (different streams) race on it -- the header tells callers to serialise them.
namespace fsk {
constexpr int kStaticPostIns = FUSEFSS_NOALLOC_MAX_INS;
// In HOST code this name is only a handle for the runtime's symbol calls, never a device address: passing it to a kernel would
// fault (or quietly use host memory where the GPU can reach it).  static_post_table() below asks the runtime for the real address.
static __device__ __align__(256) unsigned char g_static_post_ins[(size_t)kStaticPostIns * sizeof(Ins)];

namespace {
// Device address of g_static_post_ins on the CURRENT device: looked up once per device (the first noalloc call there, with that
// device current), cached afterwards.  The map node is host memory; no device allocation happens here.
int static_post_table(Ins **out) {
    static std::mutex mu;
    static std::map<int, Ins *> addr;
    int dev = 0;
    CU(cudaGetDevice(&dev));
    std::lock_guard<std::mutex> lock(mu);
    auto it = addr.find(dev);
    if (it == addr.end()) {
        void *p = nullptr;
        CU(cudaGetSymbolAddress(&p, g_static_post_ins));
        if (!p) return cuda_fail(cudaErrorInvalidSymbol, "cudaGetSymbolAddress(g_static_post_ins) returned null");
        it = addr.emplace(dev, static_cast<Ins *>(p)).first;
    }
    *out = it->second;
    return 0;
}
}  // namespace
}  // namespace fsk

extern "C" int fusefss_post_fused_noalloc(const fusefss_program *prog, const void *key0_dev, const void *key1_dev,
                                          const uint64_t *xhat_dev, const uint64_t *bits0_dev, const uint64_t *bits1_dev,
                                          const uint64_t *coeff0_dev, const uint64_t *coeff1_dev, size_t count, uint64_t *y0_dev,
                                          uint64_t *y1_dev, uint64_t *z0_dev, uint64_t *z1_dev, void *stream) {
    const Program *P = prog_of(prog);
    if (!P || !key0_dev || !key1_dev || !xhat_dev) return FUSEFSS_E_NULL;
    // the size limit is checked before anything touches the GPU (and before `count`), so a caller can probe it at start-up
    if (P->ins.size() > (size_t)kStaticPostIns) return FUSEFSS_E_STATIC;
    if (count == 0) return FUSEFSS_E_COUNT;
    if ((P->T > 0 && (!bits0_dev || !bits1_dev)) || (P->has_lut && (!coeff0_dev || !coeff1_dev))) return FUSEFSS_E_NULL;
    if ((P->n_out_a > 0 && (!y0_dev || !y1_dev)) || (P->n_out_b > 0 && (!z0_dev || !z1_dev))) return FUSEFSS_E_NULL;
    int rc = init_device(); if (rc) return rc;
    Ins *table = nullptr;
    rc = static_post_table(&table); if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    // this call's instructions -> front of the shared table, ordered before the kernel on the same stream.  P->ins is pageable host
    // memory owned by the program: the runtime has staged it by the time cudaMemcpyAsync returns, so the program may be destroyed
    // as soon as this function has returned and the stream has drained.
    if (!P->ins.empty())
        CU(cudaMemcpyAsync(table, P->ins.data(), P->ins.size() * sizeof(Ins), cudaMemcpyHostToDevice, st));
    Layout L; compute_layout(*P, count, &L);
    PostFusedArgs a{};
    a.ins = table; a.n_ins = (int)P->ins.size();
    a.mask_output = (int)P->mask_output; a.n_out_a = P->n_out_a; a.n_out_b = P->n_out_b;
    a.key[0] = (const uint8_t *)key0_dev; a.key[1] = (const uint8_t *)key1_dev; a.xhat = xhat_dev;
    a.bits[0] = bits0_dev; a.bits[1] = bits1_dev; a.coeff[0] = coeff0_dev; a.coeff[1] = coeff1_dev;
    a.y_out[0] = y0_dev; a.y_out[1] = y1_dev; a.z_out[0] = z0_dev; a.z_out[1] = z1_dev;
    a.count = count; a.mask = P->mask; a.k = post_offsets(*P, L);
    return launch_post(*P, k_post_fused<false>, k_post_fused<true>, count, st, a);
}

// ---- PRG micro-kernels: roofline denominator probe and FIPS-197 known-answer path --------------------
namespace fsk {
struct ProbeArgs { uint4 *out; size_t threads; int iters; };
__global__ void __launch_bounds__(kEvalThreads, 1) k_aes_probe(const ProbeArgs a) {
    extern __shared__ uint32_t sT[];
    const uint32_t tl = aes_fill_tables(sT);
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < a.threads; i += (size_t)gridDim.x * blockDim.x) {
        uint32_t x[1][4] = {{(uint32_t)i, (uint32_t)(i >> 32), 0x9e3779b9u, 0x7f4a7c15u}};
        for (int it = 0; it < a.iters; it += 3) {                       // 3 independent keys per trip, like a p = 3 level
            uint32_t o[1][3][4];
            prg_blocks<1, 3, 0, true>(tl, x, o);
#pragma unroll
            for (int c = 0; c < 4; ++c) x[0][c] = o[0][0][c] ^ o[0][1][(c + 1) & 3] ^ o[0][2][(c + 2) & 3];
        }
        a.out[i] = make_uint4(x[0][0], x[0][1], x[0][2], x[0][3]);
    }
}
// Pipe probes for the roofline denominators: kind 0 = LOP3 issue rate (8 independent 3-input XOR chains
// per thread), kind 1 = conflict-free LDS.32 wavefront rate (8 independent dependent-lookup chains per thread through
// the bank-replicated table, PRMT-addressed exactly like the AES lookups).
struct PipeArgs { uint32_t *out; int iters, kind; };
__global__ void __launch_bounds__(kEvalThreads, 1) k_pipe_probe(const PipeArgs a) {
    extern __shared__ uint32_t sT[];
    const uint32_t tl = aes_fill_tables(sT);
    uint32_t v[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) v[j] = threadIdx.x * 2654435761u + j * 40503u + blockIdx.x;
    if (a.kind == 0) {
        const uint32_t k1 = tl | 0x55aa55aau, k2 = tl * 3u + 1u;
        for (int i = 0; i < a.iters; ++i) {
#pragma unroll
            for (int j = 0; j < 8; ++j) asm("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(v[j]) : "r"(k1), "r"(k2 + j));
        }
    } else {
        for (int i = 0; i < a.iters; ++i) {
#pragma unroll
            for (int j = 0; j < 8; ++j) v[j] = tlu<0, 0>(tl, v[j]) + j;
        }
    }
    uint32_t acc = 0;
#pragma unroll
    for (int j = 0; j < 8; ++j) acc ^= v[j];
    a.out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = acc;
}
// Latency probe for the small-tensor floor (bench.py, DESIGN 6): ONE warp of a 256-thread CTA (the CTA size of the small evaluation kernels,
// so launch + table fill cost the same) chains `iters` dependent trips; a trip expands the lane's seed into B blocks that share their
// round-1 lookups -- the PRG work of one tree level with B blocks per node, 32 elements in lock-step -- and folds them into the next seed.
template <int B>
__global__ void __launch_bounds__(kEvalThreadsSmall, 1) k_aes_chain_probe(const ProbeArgs a) {
    extern __shared__ uint32_t sT[];
    const uint32_t tl = aes_fill_tables(sT);
    if (threadIdx.x >= 32) return;
    uint32_t x[1][4] = {{threadIdx.x * 2654435761u, 0x9e3779b9u, 0x7f4a7c15u, 0xf39cc060u}};
    for (int it = 0; it < a.iters; ++it) {
        uint32_t o[1][B][4];
        prg_blocks<1, B, 0, 1>(tl, x, o);
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            uint32_t v = 0;
#pragma unroll
            for (int k = 0; k < B; ++k) v ^= o[0][k][(c + k) & 3];
            x[0][c] = v;
        }
    }
    a.out[threadIdx.x] = make_uint4(x[0][0], x[0][1], x[0][2], x[0][3]);
}
struct KatArgs { uint4 *out; uint32_t in[4]; RoundKeys rk; };
__global__ void k_aes_kat(const KatArgs a) {
    extern __shared__ uint32_t sT[];
    const uint32_t tl = aes_fill_tables(sT);
    if (threadIdx.x == 0) {
        uint32_t s[4] = {a.in[0], a.in[1], a.in[2], a.in[3]};
        aes_encrypt_rk(tl, a.rk, s);
        a.out[0] = make_uint4(s[0], s[1], s[2], s[3]);
    }
}
}  // namespace fsk

extern "C" {

int fusefss_aes_probe(size_t threads, int iters, void *out_dev, void *stream) {
    if (!out_dev) return FUSEFSS_E_NULL;
    if (threads == 0 || iters <= 0) return FUSEFSS_E_COUNT;
    int rc = init_device(); if (rc) return rc;
    ProbeArgs a{(uint4 *)out_dev, threads, iters};
    const int grid = grid_for((threads + 31) / 32, kEvalThreads);
    return launch(k_aes_probe, grid, kEvalThreads, kAesSmemBytes, (cudaStream_t)stream, a);
}

int fusefss_aes_chain_probe(int blocks_per_trip, int trips, void *out_dev, void *stream) {
    if (!out_dev) return FUSEFSS_E_NULL;
    if (trips <= 0 || blocks_per_trip < 1 || blocks_per_trip > 5) return FUSEFSS_E_COUNT;
    int rc = init_device(); if (rc) return rc;
    ProbeArgs a{(uint4 *)out_dev, 32, trips};
    switch (blocks_per_trip) {
#define FSK_CH_CASE(BB) case BB: return launch(k_aes_chain_probe<BB>, 1, kEvalThreadsSmall, kAesSmemBytes, (cudaStream_t)stream, a);
    FSK_CH_CASE(1) FSK_CH_CASE(2) FSK_CH_CASE(3) FSK_CH_CASE(4) FSK_CH_CASE(5)
#undef FSK_CH_CASE
    }
    return FUSEFSS_E_COUNT;
}

int fusefss_pipe_probe(int kind, int iters, void *out_dev, void *stream) {
    if (!out_dev) return FUSEFSS_E_NULL;
    if (iters <= 0 || (kind != 0 && kind != 1)) return FUSEFSS_E_COUNT;
    int rc = init_device(); if (rc) return rc;
    PipeArgs a{(uint32_t *)out_dev, iters, kind};
    return launch(k_pipe_probe, g_sms, kEvalThreads, kAesSmemBytes, (cudaStream_t)stream, a);
}

// bitsliced AES core (measurement only, DESIGN 5.2): round-key bit masks -> constant memory, then the kernel
static int bitslice_upload_key(const uint8_t *key, cudaStream_t st) {
    uint32_t w[44];
    host_aes().expand(key, w);
    static thread_local uint32_t masks[11][128];
    for (int r = 0; r < 11; ++r)
        for (int b = 0; b < 16; ++b)
            for (int i = 0; i < 8; ++i) masks[r][8 * b + i] = 0u - ((w[4 * r + b / 4] >> (8 * (b % 4) + i)) & 1u);
    CU(cudaMemcpyToSymbolAsync(c_bs_rk, masks, sizeof masks, 0, cudaMemcpyHostToDevice, st));
    CU(cudaStreamSynchronize(st));
    return 0;
}

int fusefss_bitslice_kat(const uint8_t *key, const void *in_dev, void *out_dev, void *stream) {
    if (!key || !in_dev || !out_dev) return FUSEFSS_E_NULL;
    int rc = init_device(); if (rc) return rc;
    rc = bitslice_upload_key(key, (cudaStream_t)stream); if (rc) return rc;
    return launch(k_bitslice_kat, 1, 32, 0, (cudaStream_t)stream, BsKatArgs{(const uint8_t *)in_dev, (uint8_t *)out_dev});
}

int fusefss_bitslice_probe(const uint8_t *key, size_t threads, int iters, void *out_dev, void *stream) {
    if (!key || !out_dev) return FUSEFSS_E_NULL;
    if (threads == 0 || iters <= 0) return FUSEFSS_E_COUNT;
    int rc = init_device(); if (rc) return rc;
    rc = bitslice_upload_key(key, (cudaStream_t)stream); if (rc) return rc;
    const int grid = (int)std::min<size_t>((threads + 255) / 256, (size_t)g_sms * 2);
    return launch(k_bitslice_probe, grid, 256, 0, (cudaStream_t)stream, BsProbeArgs{(uint4 *)out_dev, threads, iters});
}

int fusefss_aes_kat(const uint8_t *key, const uint8_t *in, void *out_dev, void *stream) {
    if (!key || !in || !out_dev) return FUSEFSS_E_NULL;
    int rc = init_device(); if (rc) return rc;
    KatArgs a{};
    a.out = (uint4 *)out_dev;
    std::memcpy(a.in, in, 16);
    host_aes().expand(key, a.rk.w);
    return launch(k_aes_kat, 1, 256, kAesSmemBytes, (cudaStream_t)stream, a);
}

}  // extern "C"
