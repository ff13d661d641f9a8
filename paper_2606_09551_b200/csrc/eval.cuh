// eval.cuh -- online FSS evaluation kernels: packed comparison (a5) and vector interval lookup (a6).
// Def I.1: bit t = XOR share of I[view_{k_t,c_t}(xhat) < theta_t], one bit-DCF per query.
// Def I.2: additive shares of v_{i*} in R^p = c_b + sum_j vecDCF.Eval_b(key_j, xhat) (DESIGN 4.7 S2).
// DCF walk: DESIGN 4.2; PRG: DESIGN 4.1; key layout: DESIGN 4.4.
//
// Mapping: one lane per element, one warp per (32-element tile, tree group); a warp walks its trees one after
// another, the 1+Q PRG blocks of a level in lock-step.  Correction words are SoA over elements, so each level
// is one 512-B (sCW) + p 256-B (VCW) coalesced streaming load per warp, prefetched one level ahead.
#pragma once
#include "aes.cuh"

namespace fsk {

constexpr int kEvalThreads = 1024;

struct CmpAtomDev { uint64_t c; uint64_t root_off, cw_off, vb_off; int k; int pad; };
struct EvalCmpArgs {
    const uint8_t *key; const uint64_t *xhat; uint64_t *out;
    size_t count, s16;
    int T, G, party, pad;
    CmpAtomDev atom[kMaxAtoms];
};

__device__ __forceinline__ uint4 ld_stream16(const void *p) { return __ldcs(reinterpret_cast<const uint4 *>(p)); }
__device__ __forceinline__ uint64_t ld_stream8(const void *p) { return __ldcs(reinterpret_cast<const unsigned long long *>(p)); }

__global__ void __launch_bounds__(kEvalThreads, 1) k_eval_cmp(const __grid_constant__ EvalCmpArgs a) {
    extern __shared__ uint32_t sT[];
    const uint32_t tl = aes_fill_tables(sT);
    const int lane = threadIdx.x & 31;
    const size_t tiles = (a.count + 31) / 32;
    const size_t items = tiles * (size_t)a.G;
    const size_t warps = (size_t)gridDim.x * (blockDim.x >> 5);
    for (size_t it = (size_t)(threadIdx.x >> 5) * gridDim.x + blockIdx.x; it < items; it += warps) {   // warp w of CTA b takes items w*grid + b: a partial last wave spreads over all SMs
        const int g = (int)(it / tiles);
        const size_t tile = it - (size_t)g * tiles;
        size_t e = tile * 32 + lane;
        const bool live = e < a.count;
        if (!live) e = a.count - 1;
        const uint64_t xh = a.xhat[e];
        uint64_t word = 0;
        for (int t = g; t < a.T; t += a.G) {
            const CmpAtomDev &at = a.atom[t];
            const int k = at.k;
            const uint64_t km = k >= 64 ? ~0ull : ((1ull << k) - 1ull);
            uint64_t u = (((xh & km) + at.c) & km) << (64 - k);            // view_{k,c}(xhat), MSB-aligned
            uint4 s = ld_stream16(a.key + at.root_off + e * 16);
            const uint64_t vb = ld_stream8(a.key + at.vb_off + e * 8);
            const uint32_t fin = s.x & 1u;
            s.x &= ~3u;
            uint32_t tb = (uint32_t)a.party, V = 0;
            const uint8_t *cwp = a.key + at.cw_off + e * 16;
            uint4 cw = ld_stream16(cwp);
            for (int i = 0; i < k; ++i) {
                uint4 cw_next = cw;
                if (i + 1 < k) cw_next = ld_stream16(cwp + (size_t)(i + 1) * a.s16);
                const uint32_t dbit = (uint32_t)(u >> 63);
                u <<= 1;
                uint32_t x[1][4] = {{s.x | dbit, s.y, s.z, s.w}};
                uint32_t o[1][1][4];
                prg_blocks<1, 1, 0>(tl, x, o);
                const uint32_t tm = 0u - tb;                                   // all-ones iff the control bit is set
                V ^= ((o[0][0][0] >> 1) & 1u) ^ (tb & (uint32_t)((vb >> i) & 1ull));
                const uint32_t tnew = (o[0][0][0] & 1u) ^ (tb & (cw.x >> dbit) & 1u);
                s.x = (o[0][0][0] & ~3u) ^ (cw.x & ~3u & tm);
                s.y = o[0][0][1] ^ (cw.y & tm);
                s.z = o[0][0][2] ^ (cw.z & tm);
                s.w = o[0][0][3] ^ (cw.w & tm);
                tb = tnew;
                cw = cw_next;
            }
            uint32_t x[1][4] = {{s.x | 2u, s.y, s.z, s.w}};                   // leaf conversion, tweak 2
            uint32_t o[1][1][4];
            prg_blocks<1, 1, 0>(tl, x, o);
            V ^= ((o[0][0][0] >> 1) & 1u) ^ (tb & fin);
            word |= (uint64_t)(V & 1u) << t;
        }
        if (live) {
            if (a.G == 1) a.out[e] = word;
            else atomicOr(reinterpret_cast<unsigned long long *>(a.out + e), (unsigned long long)word);
        }
    }
}

struct EvalLutArgs {
    const uint8_t *key; const uint64_t *xhat; uint64_t *out;     // out[p][count]
    size_t count, s16, s8, lut_c, vt_first, vt_stride, lvl_stride, vt_lvl_rel, vt_fin_rel;
    uint64_t mask;
    int n, M, G, party;
};

template <int P>
__global__ void __launch_bounds__(kEvalThreads, 1) k_eval_lut(const __grid_constant__ EvalLutArgs a) {
    constexpr int Q = (P + 1) / 2;
    extern __shared__ uint32_t sT[];
    const uint32_t tl = aes_fill_tables(sT);
    const int lane = threadIdx.x & 31;
    const size_t tiles = (a.count + 31) / 32;
    const size_t items = tiles * (size_t)a.G;
    const size_t warps = (size_t)gridDim.x * (blockDim.x >> 5);
    for (size_t it = (size_t)(threadIdx.x >> 5) * gridDim.x + blockIdx.x; it < items; it += warps) {   // warp w of CTA b takes items w*grid + b: a partial last wave spreads over all SMs
        const int g = (int)(it / tiles);
        const size_t tile = it - (size_t)g * tiles;
        size_t e = tile * 32 + lane;
        const bool live = e < a.count;
        if (!live) e = a.count - 1;
        const uint64_t xh = (a.xhat[e] & a.mask) << (64 - a.n);
        uint64_t acc[P];
#pragma unroll
        for (int w = 0; w < P; ++w) acc[w] = g == 0 ? ld_stream8(a.key + a.lut_c + (size_t)w * a.s8 + e * 8) : 0ull;
        for (int j = 1 + g; j < a.M; j += a.G) {
            const uint8_t *tree = a.key + a.vt_first + (size_t)(j - 1) * a.vt_stride;
            uint4 s = ld_stream16(tree + e * 16);
            s.x &= ~3u;
            uint32_t tb = (uint32_t)a.party;
            uint64_t V[P];
#pragma unroll
            for (int w = 0; w < P; ++w) V[w] = 0;
            const uint8_t *lvl = tree + a.vt_lvl_rel;
            uint64_t u = xh;
            uint4 cw = ld_stream16(lvl + e * 16);
            uint64_t vcw[P];
#pragma unroll
            for (int w = 0; w < P; ++w) vcw[w] = ld_stream8(lvl + a.s16 + (size_t)w * a.s8 + e * 8);
            for (int i = 0; i < a.n; ++i) {
                lvl += a.lvl_stride;                                            // level n = the fin words: still in bounds
                uint4 cw_next = cw;
                uint64_t vcw_next[P];
                if (i + 1 < a.n) {
                    cw_next = ld_stream16(lvl + e * 16);
#pragma unroll
                    for (int w = 0; w < P; ++w) vcw_next[w] = ld_stream8(lvl + a.s16 + (size_t)w * a.s8 + e * 8);
                } else {
#pragma unroll
                    for (int w = 0; w < P; ++w) vcw_next[w] = 0;
                }
                const uint32_t dbit = (uint32_t)(u >> 63);
                u <<= 1;
                uint32_t x[1][4] = {{s.x | dbit, s.y, s.z, s.w}};
                uint32_t o[1][1 + Q][4];
                prg_blocks<1, 1 + Q, 0, true>(tl, x, o);
                const uint32_t tm = 0u - tb;
                const uint64_t tm64 = 0ull - (uint64_t)tb;
#pragma unroll
                for (int w = 0; w < P; ++w) {
                    const uint64_t W = (uint64_t)o[0][1 + w / 2][2 * (w & 1)] | ((uint64_t)o[0][1 + w / 2][2 * (w & 1) + 1] << 32);
                    V[w] += W + (vcw[w] & tm64);
                }
                const uint32_t tnew = (o[0][0][0] & 1u) ^ (tb & (cw.x >> dbit) & 1u);
                s.x = (o[0][0][0] & ~3u) ^ (cw.x & ~3u & tm);
                s.y = o[0][0][1] ^ (cw.y & tm);
                s.z = o[0][0][2] ^ (cw.z & tm);
                s.w = o[0][0][3] ^ (cw.w & tm);
                tb = tnew;
                cw = cw_next;
#pragma unroll
                for (int w = 0; w < P; ++w) vcw[w] = vcw_next[w];
            }
            // leaf: V += conv(s) + t * fin; party 1 negates
            uint32_t x[1][4] = {{s.x | 2u, s.y, s.z, s.w}};
            uint32_t o[1][Q][4];
            prg_blocks<1, Q, 1, true>(tl, x, o);
            const uint64_t tm64 = 0ull - (uint64_t)tb;
            const uint8_t *fin = tree + a.vt_fin_rel;
#pragma unroll
            for (int w = 0; w < P; ++w) {
                const uint64_t C = (uint64_t)o[0][w / 2][2 * (w & 1)] | ((uint64_t)o[0][w / 2][2 * (w & 1) + 1] << 32);
                uint64_t v = V[w] + (C & a.mask) + (ld_stream8(fin + (size_t)w * a.s8 + e * 8) & tm64);
                acc[w] += a.party ? 0ull - v : v;
            }
        }
        if (live) {
#pragma unroll
            for (int w = 0; w < P; ++w) {
                if (a.G == 1) a.out[(size_t)w * a.count + e] = acc[w] & a.mask;
                else atomicAdd(reinterpret_cast<unsigned long long *>(a.out + (size_t)w * a.count + e), (unsigned long long)acc[w]);
            }
        }
    }
}

// n < 64 with G > 1: atomics accumulate mod 2^64; reduce to the ring afterwards
struct MaskArgs { uint64_t *p; size_t words; uint64_t mask; };
__global__ void k_mask_words(const MaskArgs a) {
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < a.words) a.p[i] &= a.mask;
}

}  // namespace fsk
