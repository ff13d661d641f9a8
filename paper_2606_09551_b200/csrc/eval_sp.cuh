// eval_sp.cuh -- online evaluation for variant 1 (single-key shared-prefix construction, DESIGN.md section 9;
// SURVEY 8(f) NEXT-1; north_star: "the packed multi-threshold comparison that shares tree prefixes across the
// predicates of one element").  Per element ONE n-bit DCF key f_{r,1} (payload in R) -- plus one bit-DCF per
// narrower view -- is evaluated at the public points u_j = (xhat + delta_j) mod 2^k:
//   I[view_{k,c}(x) < beta] = e - b + a,  b = f(xhat + c), a = f(xhat + c - beta), e = I[(xhat + c) mod 2^k < beta]
// (Def I.1 with c_t = -beta_t, theta_t = r).  Predicate bits are the LSBs; the interval lookup is the
// public linear map  v_{i*} = v_{m-1} + sum_i (v_{i-1} - v_i) I[x < alpha_i]  of the same comparisons (Def I.2).
// Points whose offsets lie within 2^tail_bits of each other share the walk over their top n - tail_bits bits:
// the cluster's first candidate prefix is walked once, the second one forks off it for its last few levels
// (sp_walk_fork), every point then walks only its tail from the matching saved state.
#pragma once
#include "aes.cuh"
#include "eval.cuh"
#include "program.h"

namespace fsk {

struct SpAtomDev { uint64_t c, beta; int k, is_theta; };
struct EvalSpArgs {
    const uint8_t *key2[2]; const uint64_t *xhat; uint64_t *bits_out2[2], *coeff_out2[2];   // per party; either output may be null
    int n_parties, party0;      // 1 party (party0) or both parties in one launch (items = parties x groups x tiles)
    const SpPoint *points; const uint64_t *weights, *delta_tab, *alpha;             // device tables (program blob)
    const SpCluster *cluster;
    size_t count, s16, s8, lvl_stride, vt_first, vt_lvl_rel, vt_fin_rel, rpow;
    uint64_t mask;
    int n, m, p, et, T, n_w, n_clusters, G;     // G > 1: the points of an element are dealt round-robin to G warps (small tensors); et: early-terminated bit trees
    int zero_first, np;                         // G > 1: outputs are zeroed in-kernel before the atomics (cooperative launch); np: points per batch
    SpWidth width[kMaxWidths];
    size_t bt_root[kMaxWidths], bt_cw[kMaxWidths], bt_vb[kMaxWidths];
    SpAtomDev atom[kMaxAtoms];
};

// PK = payload words of the n-bit key: 1 (payload 1) or d+1 (payload (1, -r, .., (-r)^d), variant bit 2, DESIGN 11)
#ifndef FFS_SP_PREFETCH_BIG
#define FFS_SP_PREFETCH_BIG 0     // 1: the large-launch instantiation also prefetches the next level into registers
#endif
#ifndef FFS_SP_UNR
#define FFS_SP_UNR 3              // AES rounds per loop trip in this kernel (profiles/r1l_unroll.md)
#endif
#ifndef FFS_SP_UNR_WIDE
#define FFS_SP_UNR_WIDE FFS_SP_UNR // ... when the key's payload has >= 2 words (3 PRG blocks per level)
#endif
template <int PK> constexpr int sp_unr() { return PK >= 2 ? FFS_SP_UNR_WIDE : FFS_SP_UNR; }
template <int PK> struct SpState { uint32_t s[4]; uint32_t t; uint64_t V[PK]; };

template <int PK>
__device__ __forceinline__ void sp_step(uint32_t tl, const uint4 cw, const uint64_t (&vcw)[PK], uint32_t dbit, SpState<PK> &st) {
    constexpr int QK = (PK + 1) / 2;
    uint32_t x[1][4] = {{st.s[0] | dbit, st.s[1], st.s[2], st.s[3]}};
    uint32_t o[1][1 + QK][4];
    prg_blocks<1, 1 + QK, 0, true, sp_unr<PK>()>(tl, x, o);
    const uint32_t tm = 0u - st.t;
    const uint64_t tm64 = 0ull - (uint64_t)st.t;
#pragma unroll
    for (int w = 0; w < PK; ++w)
        st.V[w] += ((uint64_t)o[0][1 + w / 2][2 * (w & 1)] | ((uint64_t)o[0][1 + w / 2][2 * (w & 1) + 1] << 32)) + (vcw[w] & tm64);
    const uint32_t tnew = (o[0][0][0] & 1u) ^ (st.t & (cw.x >> dbit) & 1u);
    st.s[0] = (o[0][0][0] & ~3u) ^ (cw.x & ~3u & tm);
    st.s[1] = o[0][0][1] ^ (cw.y & tm);
    st.s[2] = o[0][0][2] ^ (cw.z & tm);
    st.s[3] = o[0][0][3] ^ (cw.w & tm);
    st.t = tnew;
}

// Cache behaviour of a level's correction words (HINT): the levels of a cluster's shared prefix (and every level of a lone point)
// are read exactly once per element -- streamed (ld.global.cs, evict-first); the tail levels of a cluster are re-read once per
// point of the cluster -- kept in L2 with an evict_last policy, so that the streamed prefix levels of the other 150,000 resident
// lanes do not push them out to DRAM between two points.  Measured (profiles/r2d_eval_sp_sweep.md, 1024 threads): DRAM bytes of the
// gelu launch 2.72x -> 2.15x the key, of one silu chunk 4.01x -> 2.22x.  The hints do NOT bring the kernel to 1.0x: on the final
// build profiles/traffic.md still has 2.2x on silu variant 1 and 6.5x on variant 5 (spill traffic of the 1024-thread instantiation
// plus tail levels that fall out of L2 between the points of a cluster).
#ifndef FFS_SP_L2HINT
#define FFS_SP_L2HINT 1
#endif
enum { SP_LD_PLAIN = 0, SP_LD_STREAM = 1, SP_LD_KEEP = 2 };
__device__ __forceinline__ uint64_t sp_keep_policy() {
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
template <int HINT> __device__ __forceinline__ uint4 sp_ld16(const void *p, uint64_t pol) {
    if (!FFS_SP_L2HINT || HINT == SP_LD_PLAIN) return __ldg(reinterpret_cast<const uint4 *>(p));
    if (HINT == SP_LD_STREAM) return __ldcs(reinterpret_cast<const uint4 *>(p));
    uint4 v;
    asm volatile("ld.global.nc.L2::cache_hint.v4.u32 {%0, %1, %2, %3}, [%4], %5;" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p), "l"(pol));
    return v;
}
template <int HINT> __device__ __forceinline__ uint64_t sp_ld8(const void *p, uint64_t pol) {
    if (!FFS_SP_L2HINT || HINT == SP_LD_PLAIN) return __ldg(reinterpret_cast<const unsigned long long *>(p));
    if (HINT == SP_LD_STREAM) return __ldcs(reinterpret_cast<const unsigned long long *>(p));
    uint64_t v;
    asm volatile("ld.global.nc.L2::cache_hint.u64 %0, [%1], %2;" : "=l"(v) : "l"(p), "l"(pol));
    return v;
}
template <int PK, int HINT = SP_LD_PLAIN>
__device__ __forceinline__ void sp_load_level(const uint8_t *pl, size_t e, size_t s16, size_t s8, uint4 &cw, uint64_t (&vcw)[PK], uint64_t pol = 0) {
    cw = sp_ld16<HINT>(pl + e * 16, pol);
#pragma unroll
    for (int w = 0; w < PK; ++w) vcw[w] = sp_ld8<HINT>(pl + s16 + (size_t)w * s8 + e * 8, pol);
}

// The two candidate prefixes u1, u2 of a cluster (top kf bits) usually differ only in their last few bits: walk u1
// once, snapshot the state at the level where u2 leaves u1's path (per lane), then walk u2's few remaining levels.
// On return a / b = the states after kf levels along u1 / u2 (b = a when the prefixes are equal).
template <int PK>
__device__ __forceinline__ void sp_walk_fork(uint32_t tl, const uint8_t *lvl, size_t e, size_t s16, size_t s8, size_t lvl_stride,
                                             int kf, uint64_t u1, uint64_t u2, SpState<PK> &a, SpState<PK> &b) {
    const uint64_t diff = (u1 ^ u2) >> (64 - kf);
    const int ldiv = diff ? kf - (64 - __clzll((long long)diff)) : kf;       // first level at which the prefixes differ
    const uint8_t *pl = lvl;
    uint64_t ub = u1;
    for (int i = 0; i < kf; ++i, pl += lvl_stride) {
        if (i == ldiv) b = a;
        uint4 cw; uint64_t vcw[PK];
        sp_load_level<PK, SP_LD_STREAM>(pl, e, s16, s8, cw, vcw);
        sp_step<PK>(tl, cw, vcw, (uint32_t)(ub >> 63), a);
        ub <<= 1;
    }
    if (ldiv >= kf) { b = a; return; }
    ub = u2 << ldiv;
    pl = lvl + (size_t)ldiv * lvl_stride;
    for (int i = ldiv; i < kf; ++i, pl += lvl_stride) {                       // per-lane trip count (expected ~2 levels)
        uint4 cw; uint64_t vcw[PK];
        sp_load_level<PK, SP_LD_STREAM>(pl, e, s16, s8, cw, vcw);
        sp_step<PK>(tl, cw, vcw, (uint32_t)(ub >> 63), b);
        ub <<= 1;
    }
}

// leaf: A = (-1)^party (V + conv(s) + t * fin)
template <int PK>
__device__ __forceinline__ void sp_leaf(uint32_t tl, const SpState<PK> &st, const uint8_t *fin, size_t e, size_t s8, int party, uint64_t (&A)[PK]) {
    constexpr int QK = (PK + 1) / 2;
    uint32_t x[1][4] = {{st.s[0] | 2u, st.s[1], st.s[2], st.s[3]}};
    uint32_t o[1][QK][4];
    prg_blocks<1, QK, 1, true, sp_unr<PK>()>(tl, x, o);
    const uint64_t tm64 = 0ull - (uint64_t)st.t;
#pragma unroll
    for (int w = 0; w < PK; ++w) {
        const uint64_t f = __ldg(reinterpret_cast<const unsigned long long *>(fin + (size_t)w * s8 + e * 8));
        const uint64_t v = st.V[w] + ((uint64_t)o[0][w / 2][2 * (w & 1)] | ((uint64_t)o[0][w / 2][2 * (w & 1) + 1] << 32)) + (f & tm64);
        A[w] = party ? 0ull - v : v;
    }
}

// NP points in lock-step over levels [from, to): every level's correction words are loaded ONCE for the NP points (they walk
// the same levels of the same element's key), and the NP x (1 + QK) PRG blocks of a level are NP x (1+QK) x 16 independent
// lookups per round -- the instruction-level parallelism a launch with only a few warps per SM lives on.  The next level's
// words are prefetched into registers while the current level's AES runs.
template <int PK, int NPMAX, int NP, int HINT>
__device__ __forceinline__ void sp_walk_batch(uint32_t tl, const uint8_t *lvl, size_t e, size_t s16, size_t s8, size_t lvl_stride,
                                              int from, int to, uint64_t (&ub)[NPMAX], SpState<PK> (&st)[NPMAX], uint64_t pol) {
    constexpr int QK = (PK + 1) / 2;
    // register prefetch of the next level: only where a few warps per SM must hide the load latency themselves (the 256-thread
    // instantiations, NPMAX > 1); with 32 warps per SM the other warps hide it and the 10 registers are better spent on the AES state
    constexpr bool PF = NPMAX > 1 || FFS_SP_PREFETCH_BIG;
    if (from >= to) return;
    const uint8_t *pl = lvl + (size_t)from * lvl_stride;
    uint4 cw; uint64_t vcw[PK];
    if (PF) sp_load_level<PK, HINT>(pl, e, s16, s8, cw, vcw, pol);
    for (int i = from; i < to; ++i) {
        if (!PF) sp_load_level<PK, HINT>(pl, e, s16, s8, cw, vcw, pol);
        pl += lvl_stride;
        uint4 cw_n = cw; uint64_t vcw_n[PK];
#pragma unroll
        for (int w = 0; w < PK; ++w) vcw_n[w] = vcw[w];
        if (PF && i + 1 < to) sp_load_level<PK, HINT>(pl, e, s16, s8, cw_n, vcw_n, pol);
        uint32_t x[NP][4], o[NP][1 + QK][4], dbit[NP];
#pragma unroll
        for (int q = 0; q < NP; ++q) {
            dbit[q] = (uint32_t)(ub[q] >> 63);
            ub[q] <<= 1;
            x[q][0] = st[q].s[0] | dbit[q]; x[q][1] = st[q].s[1]; x[q][2] = st[q].s[2]; x[q][3] = st[q].s[3];
        }
        prg_blocks<NP, 1 + QK, 0, 2, sp_unr<PK>()>(tl, x, o);
#pragma unroll
        for (int q = 0; q < NP; ++q) {
            const uint32_t tm = 0u - st[q].t;
            const uint64_t tm64 = 0ull - (uint64_t)st[q].t;
#pragma unroll
            for (int w = 0; w < PK; ++w)
                st[q].V[w] += ((uint64_t)o[q][1 + w / 2][2 * (w & 1)] | ((uint64_t)o[q][1 + w / 2][2 * (w & 1) + 1] << 32)) + (vcw[w] & tm64);
            const uint32_t tnew = (o[q][0][0] & 1u) ^ (st[q].t & (cw.x >> dbit[q]) & 1u);
            st[q].s[0] = (o[q][0][0] & ~3u) ^ (cw.x & ~3u & tm);
            st[q].s[1] = o[q][0][1] ^ (cw.y & tm);
            st[q].s[2] = o[q][0][2] ^ (cw.z & tm);
            st[q].s[3] = o[q][0][3] ^ (cw.w & tm);
            st[q].t = tnew;
        }
        cw = cw_n;
#pragma unroll
        for (int w = 0; w < PK; ++w) vcw[w] = vcw_n[w];
    }
}

// the first nb of the NPMAX entries (nb is warp-uniform)
template <int PK, int NPMAX, int HINT>
__device__ __forceinline__ void sp_walk_some(int nb, uint32_t tl, const uint8_t *lvl, size_t e, size_t s16, size_t s8, size_t lvl_stride,
                                             int from, int to, uint64_t (&ub)[NPMAX], SpState<PK> (&st)[NPMAX], uint64_t pol) {
    if (NPMAX >= 4 && nb == 4) sp_walk_batch<PK, NPMAX, (NPMAX >= 4 ? 4 : 1), HINT>(tl, lvl, e, s16, s8, lvl_stride, from, to, ub, st, pol);
    else if (NPMAX >= 3 && nb == 3) sp_walk_batch<PK, NPMAX, (NPMAX >= 3 ? 3 : 1), HINT>(tl, lvl, e, s16, s8, lvl_stride, from, to, ub, st, pol);
    else if (NPMAX >= 2 && nb == 2) sp_walk_batch<PK, NPMAX, (NPMAX >= 2 ? 2 : 1), HINT>(tl, lvl, e, s16, s8, lvl_stride, from, to, ub, st, pol);
    else sp_walk_batch<PK, NPMAX, 1, HINT>(tl, lvl, e, s16, s8, lvl_stride, from, to, ub, st, pol);
}

#ifndef FFS_SP_THREADS
#define FFS_SP_THREADS 1024      // CTA size of the large launches of k_eval_sp (registers per thread = 65536 / this)
#endif
#ifndef FFS_SP_NP_BIG
#define FFS_SP_NP_BIG 1          // points walked in lock-step by the large-launch instantiation
#endif
constexpr int kEvalSpThreads = FFS_SP_THREADS;
#ifndef FFS_SP_NP_SMALL
#define FFS_SP_NP_SMALL 2        // ... by the 256-thread instantiation (255 registers per thread)
#endif

template <int P, int PK, int THREADS>
__global__ void __launch_bounds__(THREADS, 1) k_eval_sp(const __grid_constant__ EvalSpArgs a) {
    extern __shared__ uint32_t sT[];
    const uint32_t tl = aes_fill_tables(sT);
    const uint64_t keep_pol = sp_keep_policy();
    if (a.zero_first) zero_outputs_and_sync(a.bits_out2, true, a.coeff_out2, true, a.count, P);
    const size_t tiles = (a.count + 31) / 32, items = tiles * (size_t)a.G * (size_t)a.n_parties, warps = (size_t)gridDim.x * (blockDim.x >> 5);
    // warp w of CTA b takes items w*grid + b (+ k*warps): a partial last wave spreads evenly over all SMs
    for (size_t item = (size_t)(threadIdx.x >> 5) * gridDim.x + blockIdx.x; item < items; item += warps) {
        const int pg = (int)(item / tiles);                                 // (party slot, group): warp-uniform
        const size_t tile = item - (size_t)pg * tiles;
        const int slot = pg / a.G, g = pg - slot * a.G;                     // g = this warp's share of every element's points
        const int party = a.n_parties == 2 ? slot : a.party0;
        const uint8_t *key = a.key2[slot];
        uint64_t *bits_out = a.bits_out2[slot], *coeff_out = a.coeff_out2[slot];
        const size_t e0 = tile * 32 + (threadIdx.x & 31);
        const bool live = e0 < a.count;
        const size_t e = live ? e0 : a.count - 1;
        const uint64_t xh = a.xhat[e] & a.mask;
        const bool want_bits = bits_out != nullptr, want_coeff = coeff_out != nullptr;
        uint64_t word = 0, acc[P];
#pragma unroll
        for (int w = 0; w < P; ++w) acc[w] = 0;
        if (party == 0 && g == 0) {                                       // public parts: e_t and the plaintext table row of xhat
            if (want_bits)
                for (int t = 0; t < a.T; ++t) {
                    const SpAtomDev &at = a.atom[t];
                    const uint64_t km = at.k >= 64 ? ~0ull : ((1ull << at.k) - 1ull);
                    if (at.is_theta) word |= (uint64_t)(((xh + at.c) & km) < at.beta) << t;
                }
        }
        if (want_coeff && g == 0) {                                         // sum_t [(-r)^t] (w_{m-1} + sum_{i: xhat < alpha_i} (w_{i-1} - w_i))
            uint64_t rp[PK];
            rp[0] = party == 0 ? 1ull : 0ull;
#pragma unroll
            for (int t = 1; t < PK; ++t) rp[t] = __ldg(reinterpret_cast<const unsigned long long *>(key + a.rpow + (size_t)(t - 1) * a.s8 + e * 8));
            if (PK > 1 || party == 0) {
                for (int i = 0; i < a.m; ++i)
                    if (i == 0 || xh < a.alpha[i - 1]) {
#pragma unroll
                        for (int w = 0; w < P; ++w)
#pragma unroll
                            for (int t = 0; t < PK; ++t) acc[w] += a.delta_tab[((size_t)i * P + w) * PK + t] * rp[t];
                    }
            }
        }
        for (int wd = 0; wd < a.n_w; ++wd) {
            const SpWidth W = a.width[wd];
            const SpPoint *pts = a.points + W.first_point;
            const uint64_t *wts = a.weights + (size_t)W.first_point * P * PK;
            if (!W.is_vec) {
                if (!want_bits) continue;
                const uint64_t km = (1ull << W.k) - 1ull;
                for (int j = g; j < W.n_points; j += a.G) {
                    const uint64_t u = (((xh & km) + pts[j].delta) & km) << (64 - W.k);
                    const uint32_t A = bit_tree_eval<false>(tl, key, a.bt_root[wd], a.bt_cw[wd], a.bt_vb[wd], e, a.s16, W.k, u, party, a.et);
                    word ^= pts[j].bitmask & (0ull - (uint64_t)A);
                }
                continue;
            }
            const uint8_t *tree = key + a.vt_first;
            const uint8_t *lvl = tree + a.vt_lvl_rel;
            if (a.G > 1) {                                                   // small tensors: too few warps to hide DRAM latency level by level,
                for (int i = 0; i < a.n; ++i) {                              // so pull the element's correction words towards L2 up front
                    const uint8_t *pl = lvl + (size_t)i * a.lvl_stride;
                    asm volatile("prefetch.global.L2 [%0];" ::"l"(pl + e * 16));
                    asm volatile("prefetch.global.L2 [%0];" ::"l"(pl + a.s16 + e * 8));
                }
            }
            const uint4 root = __ldg(reinterpret_cast<const uint4 *>(tree + e * 16));
            const uint8_t *fin = tree + a.vt_fin_rel;
            SpState<PK> r0;
            r0.s[0] = root.x & ~3u; r0.s[1] = root.y; r0.s[2] = root.z; r0.s[3] = root.w; r0.t = (uint32_t)party;
#pragma unroll
            for (int t = 0; t < PK; ++t) r0.V[t] = 0;
            const int n = a.n;
            constexpr int NP = THREADS == kEvalThreadsSmall ? FFS_SP_NP_SMALL : FFS_SP_NP_BIG;
            const int np = a.np < 1 ? 1 : a.np > NP ? NP : a.np;           // points walked in lock-step (<= NP, the compiled maximum)
            // is point j needed by the outputs this launch produces?  (warp-uniform)
            auto needed = [&](int j) {
                bool need = want_bits && pts[j].bitmask != 0;
                if (want_coeff) {
#pragma unroll
                    for (int w = 0; w < P * PK; ++w) need = need || wts[(size_t)j * P * PK + w] != 0;
                }
                return need;
            };
            // leaf of a walked point: A_j = share of (1, -r, ..) I[u_j < r]; fold it into the outputs
            auto fold = [&](int j, const SpState<PK> &st) {
                uint64_t A[PK];
                sp_leaf<PK>(tl, st, fin, e, a.s8, party, A);
                word ^= pts[j].bitmask & (0ull - (A[0] & 1ull));            // component 0 = share of I[u_j < r]
                if (want_coeff) {
#pragma unroll
                    for (int w = 0; w < P; ++w)
#pragma unroll
                        for (int t = 0; t < PK; ++t) acc[w] += wts[((size_t)j * P + w) * PK + t] * A[t];
                }
            };
            // (A) clusters of one point: nothing to share; the s-th of them belongs to group s mod G; NP of them walk the whole
            //     tree in lock-step
            {
                int jq[NP], nb = 0, s_idx = 0;
                auto flush = [&]() {
                    if (!nb) return;
                    SpState<PK> st[NP]; uint64_t ub[NP];
#pragma unroll
                    for (int q = 0; q < NP; ++q) {
                        st[q] = r0;
                        ub[q] = ((xh + pts[jq[q < nb ? q : 0]].delta) & a.mask) << (64 - n);
                    }
                    sp_walk_some<PK, NP, SP_LD_STREAM>(nb, tl, lvl, e, a.s16, a.s8, a.lvl_stride, 0, n, ub, st, 0);
#pragma unroll
                    for (int q = 0; q < NP; ++q) if (q < nb) fold(jq[q], st[q]);
                    nb = 0;
                };
                for (int c = 0; c < a.n_clusters; ++c) {
                    const SpCluster cl = a.cluster[c];
                    if (cl.count > 1 && n - cl.tail_bits > 0) continue;
                    for (int j = cl.first; j < cl.first + cl.count; ++j, ++s_idx) {
                        if (s_idx % a.G != g || !needed(j)) continue;
#pragma unroll
                        for (int q = 0; q < NP; ++q) if (q == nb) jq[q] = j;
                        if (++nb == np) flush();
                    }
                }
                flush();
            }
            // (B) clusters that share a prefix: walk it once (two candidates, forked), then the tails of this group's points, NP at a time
            for (int c = 0; c < a.n_clusters; ++c) {
                const SpCluster cl = a.cluster[c];
                const int kf = n - cl.tail_bits;                            // shared levels
                if (!(cl.count > 1 && kf > 0)) continue;
                bool any = false;
                for (int j = cl.first + g; j < cl.first + cl.count; j += a.G) any = any || needed(j);
                if (!any) continue;
                SpState<PK> s1 = r0, s2 = r0;
                const uint64_t uf = ((xh + pts[cl.first].delta) & a.mask) << (64 - n);
                const uint64_t ul = ((xh + pts[cl.first + cl.count - 1].delta) & a.mask) << (64 - n);
                sp_walk_fork<PK>(tl, lvl, e, a.s16, a.s8, a.lvl_stride, kf, uf, ul, s1, s2);
                const uint64_t pre1 = uf >> (64 - kf);
                int j = cl.first + g;
                while (j < cl.first + cl.count) {
                    int jq[NP], nb = 0;
                    for (; j < cl.first + cl.count && nb < np; j += a.G) {
                        if (!needed(j)) continue;
#pragma unroll
                        for (int q = 0; q < NP; ++q) if (q == nb) jq[q] = j;
                        ++nb;
                    }
                    if (!nb) break;
                    SpState<PK> st[NP]; uint64_t ub[NP];
#pragma unroll
                    for (int q = 0; q < NP; ++q) {
                        const uint64_t u = ((xh + pts[jq[q < nb ? q : 0]].delta) & a.mask) << (64 - n);
                        st[q] = (u >> (64 - kf)) == pre1 ? s1 : s2;
                        ub[q] = u << kf;
                    }
                    sp_walk_some<PK, NP, SP_LD_KEEP>(nb, tl, lvl, e, a.s16, a.s8, a.lvl_stride, kf, n, ub, st, keep_pol);
#pragma unroll
                    for (int q = 0; q < NP; ++q) if (q < nb) fold(jq[q], st[q]);
                }
            }
        }
        if (live) {
            if (a.G == 1) {
                if (want_bits) bits_out[e] = word;
                if (want_coeff) {
#pragma unroll
                    for (int w = 0; w < P; ++w) coeff_out[(size_t)w * a.count + e] = acc[w] & a.mask;
                }
            } else {                                                        // integer xor / add: order-independent, still bit-exact
                if (want_bits) atomicXor(reinterpret_cast<unsigned long long *>(bits_out + e), (unsigned long long)word);
                if (want_coeff) {
#pragma unroll
                    for (int w = 0; w < P; ++w) atomic_add_ring(coeff_out + (size_t)w * a.count + e, acc[w] & a.mask, a.mask);
                }
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------------------------------------
// Variant bit 4 (DESIGN 14; "the dense table bit-width k (DPF-LUT representation)"): the interval lookup with the
// operator as a dense table of 2^n entries.  The single key f_{r,1} is evaluated on the WHOLE domain -- a traversal of its GGM
// tree that shares every prefix -- and  share_b = [b=0] T[xhat] + sum_v D[(xhat - v) mod N] A_b(v),  D[a] = T[a-1] - T[a],
// A_b(v) = Eval_b(key, v).  One warp per (party, element): lane l owns the subtree under the top min(5, n) bits = l, walks it
// depth-first (a node is expanded once: 2 (2^(n+1) - 2) + 2^n PRG blocks per element per party), and the 32 partial sums are
// combined with shuffles.  Work and shape depend on n only.
struct EvalDenseArgs {
    const uint8_t *key2[2]; const uint64_t *xhat; uint64_t *coeff_out2[2];
    const uint64_t *dense_t, *dense_d;
    size_t count, s16, s8, lvl_stride, vt_first, vt_lvl_rel, vt_fin_rel;
    uint64_t mask;
    int n, n_parties, party0, pad;
};

template <int P>
__global__ void __launch_bounds__(kEvalThreadsSmall, 1) k_eval_dense(const __grid_constant__ EvalDenseArgs a) {
    extern __shared__ uint32_t sT[];
    const uint32_t tl = aes_fill_tables(sT);
    const int lane = threadIdx.x & 31, n = a.n;
    const int top = n < 5 ? n : 5, m = n - top;
    const size_t items = a.count * (size_t)a.n_parties, warps = (size_t)gridDim.x * (blockDim.x >> 5);
    for (size_t item = (size_t)(threadIdx.x >> 5) * gridDim.x + blockIdx.x; item < items; item += warps) {
        const int slot = (int)(item / a.count);
        const size_t e = item - (size_t)slot * a.count;
        const int party = a.n_parties == 2 ? slot : a.party0;
        const uint8_t *tree = a.key2[slot] + a.vt_first, *lvl = tree + a.vt_lvl_rel, *fin = tree + a.vt_fin_rel;
        const uint64_t xh = a.xhat[e] & a.mask;
        const bool active = lane < (1 << top);
        const uint32_t sub = active ? (uint32_t)lane : 0u;                 // idle lanes (n < 5) shadow lane 0 and contribute nothing
        const uint4 root = __ldg(reinterpret_cast<const uint4 *>(tree + e * 16));
        SpState<1> stack[12];                                              // stack[l] = the node after top + l levels (m <= 11)
        stack[0].s[0] = root.x & ~3u; stack[0].s[1] = root.y; stack[0].s[2] = root.z; stack[0].s[3] = root.w;
        stack[0].t = (uint32_t)party; stack[0].V[0] = 0;
        for (int i = 0; i < top; ++i) {                                    // this lane's path through the top levels
            uint4 cw; uint64_t vcw[1];
            sp_load_level<1>(lvl + (size_t)i * a.lvl_stride, e, a.s16, a.s8, cw, vcw);
            sp_step<1>(tl, cw, vcw, (sub >> (top - 1 - i)) & 1u, stack[0]);
        }
        uint64_t acc[P];
#pragma unroll
        for (int w = 0; w < P; ++w) acc[w] = 0;
        for (uint32_t j = 0; j < (1u << m); ++j) {                        // leaves of the subtree, left to right
            const int L = j == 0 ? 0 : m - 1 - (__ffs((int)j) - 1);       // first level whose node changes: the bit that flipped to 1
            for (int l = L; l < m; ++l) {
                uint4 cw; uint64_t vcw[1];
                sp_load_level<1>(lvl + (size_t)(top + l) * a.lvl_stride, e, a.s16, a.s8, cw, vcw);
                SpState<1> st = stack[l];
                sp_step<1>(tl, cw, vcw, (j >> (m - 1 - l)) & 1u, st);
                stack[l + 1] = st;
            }
            uint64_t A[1];
            sp_leaf<1>(tl, stack[m], fin, e, a.s8, party, A);
            const uint64_t v = ((uint64_t)sub << m) | j;
            const uint64_t *d = a.dense_d + (size_t)((xh - v) & a.mask) * P;
#pragma unroll
            for (int w = 0; w < P; ++w) acc[w] += __ldg(d + w) * A[0];
        }
#pragma unroll
        for (int w = 0; w < P; ++w) {
            uint64_t s = active ? acc[w] : 0ull;
#pragma unroll
            for (int off = 16; off > 0; off >>= 1) s += __shfl_xor_sync(0xffffffffu, s, off);
            if (lane == 0) a.coeff_out2[slot][(size_t)w * a.count + e] = (s + (party == 0 ? __ldg(a.dense_t + (size_t)xh * P + w) : 0ull)) & a.mask;
        }
    }
}

}  // namespace fsk
