// eval_sp_split.cuh -- k_eval_sp for SMALL launches (a few thousand elements: relu16, recip, rsqrt in the single-key construction).
// A lone warp per scheduler is bound by its own instruction stream (about 1,000 instructions per level when one lane expands the
// child block and the payload blocks of a level: measured 1 us per level, profiles/r2u_small_split.md).  Here the 1 + QK PRG blocks
// of a level are dealt to the LANES of a group: lane k = 0 of an element's group expands the child block (key K_0), lane k >= 1 the
// payload block k - 1 (key K_k) and keeps the two accumulator words that block feeds; the child lane's new seed and control bit go
// to the group by shuffles.  A warp then carries 32 / L elements (L = 2 lanes per element for a one-block payload, 4 for two blocks)
// and executes ONE block's instructions per level, so the same tensor runs on twice (four times) as many warps with the same total
// work -- more warps per scheduler to hide each other's dependency stalls.  Same arithmetic, same outputs as k_eval_sp (DESIGN 9).
// The lane's PRG key is a run-time choice, so the expanded round keys sit in shared memory (the unused head of the table window).
#pragma once
#include "eval_sp.cuh"

namespace fsk {

struct SpL { uint32_t s[4]; uint32_t t; uint64_t V0, V1; };     // replicated seed / control bit; this lane's two accumulator words

// round keys of K_0 .. K_4 in shared memory: word 44 i + j (they start at offset 0 of the dynamic window, below the tables)
__device__ __forceinline__ void split_fill_keys(uint32_t *dyn_smem) {
    for (int i = threadIdx.x; i < kNumPrgKeys * 44; i += blockDim.x) dyn_smem[i] = c_rk[i / 44][i % 44];
    __syncthreads();
}

// PRG_k(x) = AES_{K_k}(x) ^ x with the round keys read from shared memory (rk = this lane's key)
__device__ __forceinline__ void prg_rt(uint32_t tl, const uint32_t *rk, const uint32_t (&x)[4], uint32_t (&o)[4]) {
    uint32_t s[4];
#pragma unroll
    for (int c = 0; c < 4; ++c) s[c] = x[c] ^ rk[c];
#pragma unroll 3
    for (int r = 1; r < 10; ++r) aes_round(s, tl, rk[4 * r], rk[4 * r + 1], rk[4 * r + 2], rk[4 * r + 3]);
    aes_last(s, tl, rk[40], rk[41], rk[42], rk[43]);
#pragma unroll
    for (int c = 0; c < 4; ++c) o[c] = s[c] ^ x[c];
}

// one level: every lane expands its own block of the common seed; payload lanes accumulate, the child lane's result is broadcast
__device__ __forceinline__ void split_step(uint32_t tl, const uint32_t *rk, int base, const uint4 cw, uint64_t vcw0, uint64_t vcw1,
                                           uint32_t dbit, SpL &st) {
    uint32_t x[4] = {st.s[0] | dbit, st.s[1], st.s[2], st.s[3]}, o[4];
    prg_rt(tl, rk, x, o);
    const uint32_t tm = 0u - st.t;
    const uint64_t tm64 = 0ull - (uint64_t)st.t;
    st.V0 += ((uint64_t)o[0] | ((uint64_t)o[1] << 32)) + (vcw0 & tm64);      // meaningful in payload lanes only
    st.V1 += ((uint64_t)o[2] | ((uint64_t)o[3] << 32)) + (vcw1 & tm64);
    const uint32_t tnew = (o[0] & 1u) ^ (st.t & (cw.x >> dbit) & 1u);      // meaningful in the child lane only
    const uint32_t n0 = (o[0] & ~3u) ^ (cw.x & ~3u & tm), n1 = o[1] ^ (cw.y & tm), n2 = o[2] ^ (cw.z & tm), n3 = o[3] ^ (cw.w & tm);
    st.s[0] = __shfl_sync(0xffffffffu, n0, base);
    st.s[1] = __shfl_sync(0xffffffffu, n1, base);
    st.s[2] = __shfl_sync(0xffffffffu, n2, base);
    st.s[3] = __shfl_sync(0xffffffffu, n3, base);
    st.t = __shfl_sync(0xffffffffu, tnew, base);
}

// levels [from, to) of the n-bit tree; w0 / w1 = the payload words this lane accumulates (clamped to a valid word for the child lane)
__device__ __forceinline__ void split_walk(uint32_t tl, const uint32_t *rk, int base, const uint8_t *lvl, size_t e, size_t s16, size_t s8,
                                           size_t lvl_stride, int w0, int w1, int from, int to, uint64_t ubits, SpL &st) {
    const uint8_t *pl = lvl + (size_t)from * lvl_stride;
    for (int i = from; i < to; ++i, pl += lvl_stride) {
        const uint4 cw = __ldg(reinterpret_cast<const uint4 *>(pl + e * 16));
        const uint64_t v0 = __ldg(reinterpret_cast<const unsigned long long *>(pl + s16 + (size_t)w0 * s8 + e * 8));
        const uint64_t v1 = __ldg(reinterpret_cast<const unsigned long long *>(pl + s16 + (size_t)w1 * s8 + e * 8));
        split_step(tl, rk, base, cw, v0, v1, (uint32_t)(ubits >> 63), st);
        ubits <<= 1;
    }
}

template <int P, int PK>
__global__ void __launch_bounds__(kEvalThreadsSmall, 1) k_eval_sp_split(const __grid_constant__ EvalSpArgs a) {
    constexpr int QK = (PK + 1) / 2, L = QK == 1 ? 2 : 4, EPW = 32 / L;
    constexpr unsigned FULL = 0xffffffffu;
    extern __shared__ uint32_t sT[];
    const uint32_t tl = aes_fill_tables(sT);
    split_fill_keys(sT);
    if (a.zero_first) zero_outputs_and_sync(a.bits_out2, true, a.coeff_out2, true, a.count, P);
    const int lane = threadIdx.x & 31, k = lane % L, base = lane - k;
    const int kk = k <= QK ? k : 0;                                          // a spare lane (L = 4, QK = 2) shadows the child lane
    const uint32_t *rk = sT + 44 * kk;
    const int w0 = kk >= 1 ? (2 * (kk - 1) < PK ? 2 * (kk - 1) : PK - 1) : 0;               // this lane's payload words (clamped: a valid address)
    const int w1 = kk >= 1 ? (2 * (kk - 1) + 1 < PK ? 2 * (kk - 1) + 1 : PK - 1) : 0;
    const size_t tiles = (a.count + EPW - 1) / EPW, items = tiles * (size_t)a.G * (size_t)a.n_parties, warps = (size_t)gridDim.x * (blockDim.x >> 5);
    for (size_t item = (size_t)(threadIdx.x >> 5) * gridDim.x + blockIdx.x; item < items; item += warps) {
        const int pg = (int)(item / tiles);
        const size_t tile = item - (size_t)pg * tiles;
        const int slot = pg / a.G, g = pg - slot * a.G;
        const int party = a.n_parties == 2 ? slot : a.party0;
        const uint8_t *key = a.key2[slot];
        uint64_t *bits_out = a.bits_out2[slot], *coeff_out = a.coeff_out2[slot];
        const size_t e0 = tile * EPW + (size_t)(lane / L);
        const bool live = e0 < a.count;
        const size_t e = live ? e0 : a.count - 1;                            // dead groups shadow the last element and store nothing
        const uint64_t xh = a.xhat[e] & a.mask;
        const bool want_bits = bits_out != nullptr, want_coeff = coeff_out != nullptr;
        uint64_t word = 0, acc[P];                                           // replicated in the lanes of a group; the leader stores
#pragma unroll
        for (int w = 0; w < P; ++w) acc[w] = 0;
        if (party == 0 && g == 0 && want_bits)
            for (int t = 0; t < a.T; ++t) {
                const SpAtomDev &at = a.atom[t];
                const uint64_t km = at.k >= 64 ? ~0ull : ((1ull << at.k) - 1ull);
                if (at.is_theta) word |= (uint64_t)(((xh + at.c) & km) < at.beta) << t;
            }
        if (want_coeff && g == 0) {
            uint64_t rp[PK];
            rp[0] = party == 0 ? 1ull : 0ull;
#pragma unroll
            for (int t = 1; t < PK; ++t) rp[t] = __ldg(reinterpret_cast<const unsigned long long *>(key + a.rpow + (size_t)(t - 1) * a.s8 + e * 8));
            if (PK > 1 || party == 0)
                for (int i = 0; i < a.m; ++i)
                    if (i == 0 || xh < a.alpha[i - 1]) {
#pragma unroll
                        for (int w = 0; w < P; ++w)
#pragma unroll
                            for (int t = 0; t < PK; ++t) acc[w] += a.delta_tab[((size_t)i * P + w) * PK + t] * rp[t];
                    }
        }
        for (int wd = 0; wd < a.n_w; ++wd) {
            const SpWidth W = a.width[wd];
            const SpPoint *pts = a.points + W.first_point;
            const uint64_t *wts = a.weights + (size_t)W.first_point * P * PK;
            if (!W.is_vec) {                                                 // narrower bit trees: one block per level anyway; the group's lanes agree
                if (!want_bits) continue;
                const uint64_t km = (1ull << W.k) - 1ull;
                for (int j = g; j < W.n_points; j += a.G) {
                    const uint64_t u = (((xh & km) + pts[j].delta) & km) << (64 - W.k);
                    const uint32_t A = bit_tree_eval<false>(tl, key, a.bt_root[wd], a.bt_cw[wd], a.bt_vb[wd], e, a.s16, W.k, u, party, a.et);
                    word ^= pts[j].bitmask & (0ull - (uint64_t)A);
                }
                continue;
            }
            const uint8_t *tree = key + a.vt_first, *lvl = tree + a.vt_lvl_rel, *fin = tree + a.vt_fin_rel;
            const int n = a.n;
            for (int i = 0; i < n; ++i) {                                    // pull the element's correction words towards L2 up front
                const uint8_t *pl = lvl + (size_t)i * a.lvl_stride;
                asm volatile("prefetch.global.L2 [%0];" ::"l"(pl + e * 16));
                asm volatile("prefetch.global.L2 [%0];" ::"l"(pl + a.s16 + e * 8));
            }
            const uint4 root = __ldg(reinterpret_cast<const uint4 *>(tree + e * 16));
            SpL r0;
            r0.s[0] = root.x & ~3u; r0.s[1] = root.y; r0.s[2] = root.z; r0.s[3] = root.w; r0.t = (uint32_t)party; r0.V0 = 0; r0.V1 = 0;
            auto needed = [&](int j) {                                       // warp-uniform
                bool need = want_bits && pts[j].bitmask != 0;
                if (want_coeff) {
#pragma unroll
                    for (int w = 0; w < P * PK; ++w) need = need || wts[(size_t)j * P * PK + w] != 0;
                }
                return need;
            };
            // leaf of a walked point: the payload lanes convert their block, A[t] = share of (1, -r, ..)[t] I[u_j < r] is gathered by shuffles
            auto fold = [&](int j, const SpL &st) {
                uint32_t x[4] = {st.s[0] | 2u, st.s[1], st.s[2], st.s[3]}, o[4];
                prg_rt(tl, rk, x, o);
                const uint64_t tm64 = 0ull - (uint64_t)st.t;
                const uint64_t f0 = __ldg(reinterpret_cast<const unsigned long long *>(fin + (size_t)w0 * a.s8 + e * 8));
                const uint64_t f1 = __ldg(reinterpret_cast<const unsigned long long *>(fin + (size_t)w1 * a.s8 + e * 8));
                uint64_t a0 = st.V0 + ((uint64_t)o[0] | ((uint64_t)o[1] << 32)) + (f0 & tm64);
                uint64_t a1 = st.V1 + ((uint64_t)o[2] | ((uint64_t)o[3] << 32)) + (f1 & tm64);
                if (party) { a0 = 0ull - a0; a1 = 0ull - a1; }
                uint64_t A[PK];
#pragma unroll
                for (int t = 0; t < PK; ++t) A[t] = __shfl_sync(FULL, (t & 1) ? a1 : a0, base + 1 + t / 2);
                word ^= pts[j].bitmask & (0ull - (A[0] & 1ull));
                if (want_coeff) {
#pragma unroll
                    for (int w = 0; w < P; ++w)
#pragma unroll
                        for (int t = 0; t < PK; ++t) acc[w] += wts[((size_t)j * P + w) * PK + t] * A[t];
                }
            };
            // (A) clusters of one point: the s-th of them belongs to group s mod G
            int s_idx = 0;
            for (int c = 0; c < a.n_clusters; ++c) {
                const SpCluster cl = a.cluster[c];
                if (cl.count > 1 && n - cl.tail_bits > 0) continue;
                for (int j = cl.first; j < cl.first + cl.count; ++j, ++s_idx) {
                    if (s_idx % a.G != g || !needed(j)) continue;
                    SpL st = r0;
                    split_walk(tl, rk, base, lvl, e, a.s16, a.s8, a.lvl_stride, w0, w1, 0, n, ((xh + pts[j].delta) & a.mask) << (64 - n), st);
                    fold(j, st);
                }
            }
            // (B) clusters with a shared prefix: first candidate prefix once, the second forked off it, then this group's tails
            for (int c = 0; c < a.n_clusters; ++c) {
                const SpCluster cl = a.cluster[c];
                const int kf = n - cl.tail_bits;
                if (!(cl.count > 1 && kf > 0)) continue;
                bool any = false;
                for (int j = cl.first + g; j < cl.first + cl.count; j += a.G) any = any || needed(j);
                if (!any) continue;
                const uint64_t uf = ((xh + pts[cl.first].delta) & a.mask) << (64 - n);
                const uint64_t ul = ((xh + pts[cl.first + cl.count - 1].delta) & a.mask) << (64 - n);
                const uint64_t diff = (uf ^ ul) >> (64 - kf);
                const int ldiv = diff ? kf - (64 - __clzll((long long)diff)) : kf;  // first level at which the prefixes differ (same in a group)
                const int lmin = __reduce_min_sync(FULL, ldiv);                     // the re-walk below must stay warp-uniform (shuffles inside)
                SpL s1 = r0, s2 = r0;
                {
                    const uint8_t *pl = lvl;
                    uint64_t ub = uf;
                    for (int i = 0; i < kf; ++i, pl += a.lvl_stride) {
                        if (i == ldiv) s2 = s1;
                        const uint4 cw = __ldg(reinterpret_cast<const uint4 *>(pl + e * 16));
                        const uint64_t v0 = __ldg(reinterpret_cast<const unsigned long long *>(pl + a.s16 + (size_t)w0 * a.s8 + e * 8));
                        const uint64_t v1 = __ldg(reinterpret_cast<const unsigned long long *>(pl + a.s16 + (size_t)w1 * a.s8 + e * 8));
                        split_step(tl, rk, base, cw, v0, v1, (uint32_t)(ub >> 63), s1);
                        ub <<= 1;
                    }
                    if (ldiv >= kf) s2 = s1;
                    pl = lvl + (size_t)lmin * a.lvl_stride;
                    for (int i = lmin; i < kf; ++i, pl += a.lvl_stride) {      // groups whose fork lies deeper idle through their first trips
                        const uint4 cw = __ldg(reinterpret_cast<const uint4 *>(pl + e * 16));
                        const uint64_t v0 = __ldg(reinterpret_cast<const unsigned long long *>(pl + a.s16 + (size_t)w0 * a.s8 + e * 8));
                        const uint64_t v1 = __ldg(reinterpret_cast<const unsigned long long *>(pl + a.s16 + (size_t)w1 * a.s8 + e * 8));
                        SpL tmp = s2;
                        split_step(tl, rk, base, cw, v0, v1, (uint32_t)((ul >> (63 - i)) & 1ull), tmp);
                        if (i >= ldiv) s2 = tmp;
                    }
                }
                const uint64_t pre1 = uf >> (64 - kf);
                for (int j = cl.first + g; j < cl.first + cl.count; j += a.G) {
                    if (!needed(j)) continue;
                    const uint64_t u = ((xh + pts[j].delta) & a.mask) << (64 - n);
                    SpL st = (u >> (64 - kf)) == pre1 ? s1 : s2;
                    split_walk(tl, rk, base, lvl, e, a.s16, a.s8, a.lvl_stride, w0, w1, kf, n, u << kf, st);
                    fold(j, st);
                }
            }
        }
        if (live && k == 0) {
            if (a.G == 1) {
                if (want_bits) bits_out[e] = word;
                if (want_coeff) {
#pragma unroll
                    for (int w = 0; w < P; ++w) coeff_out[(size_t)w * a.count + e] = acc[w] & a.mask;
                }
            } else {
                if (want_bits) atomicXor(reinterpret_cast<unsigned long long *>(bits_out + e), (unsigned long long)word);
                if (want_coeff) {
#pragma unroll
                    for (int w = 0; w < P; ++w) atomic_add_ring(coeff_out + (size_t)w * a.count + e, acc[w] & a.mask, a.mask);
                }
            }
        }
    }
}

}  // namespace fsk
