// eval.cuh -- online FSS evaluation for the Protocol-3 construction: packed comparison (a5) and vector interval lookup
// (a6) in ONE kernel.
// Def I.1: bit t = XOR share of I[view_{k_t,c_t}(xhat) < theta_t], one bit-DCF per query.
// Def I.2: additive shares of v_{i*} in R^p = c_b + sum_j vecDCF.Eval_b(key_j, xhat) (DESIGN 4.7 S2).
// DCF walk: DESIGN 4.2; PRG: DESIGN 4.1; key layout: DESIGN 4.4; early-terminated bit trees: DESIGN 13.
//
// Mapping: one lane per element, one warp per work item; an item = (party slot, call, tree group g, 32-element tile).  A warp
// walks the trees g, g+G, .. of its call one after another, the 1+Q PRG blocks of a level in lock-step.  Correction words are
// SoA over elements, so each level is one 512-B (sCW) + p 256-B (VCW) coalesced streaming load per warp, prefetched one level
// ahead.  fusefss_eval_cmp / _lut / _fused / _fused_both all launch this kernel with the items they need: one party or both,
// one call or both -- so a small tensor is ONE launch ("a single batched routine (e.g., one GPU kernel launch)").
// G > 1 (the trees of an element dealt to several warps so that a small launch still fills the machine): partial results are
// combined with 64-bit atomics (integer, order-independent => still bit-exact); the outputs are zeroed inside the kernel
// first (cooperative launch, one grid-wide barrier), so no memset / fix-up launches surround it.
#pragma once
#include <cooperative_groups.h>

#include "aes.cuh"

namespace fsk {

constexpr int kEvalThreads = 1024;     // large launches: 32 warps per SM hide every latency at 64 registers per thread
// CTA size of the large k_eval_p3 launches (registers per thread = 65536 / this), chosen per payload width by measurement
// (profiles/r2f_p3_threads.md): with p >= 2 a level expands 1 + ceil(p/2) >= 2 blocks in lock-step and keeps p 64-bit accumulators and p
// correction words live -- 64 registers spill; 512 threads x 128 registers run 2-3 % faster (gelu / nexp / silu).  p = 1 (shift_relu) has
// one payload block and is faster with 32 warps.  -DFFS_P3_THREADS=N forces one size for every p.
#ifdef FFS_P3_THREADS
constexpr int p3_threads_for(int) { return FFS_P3_THREADS; }
#else
constexpr int p3_threads_for(int p) { return p >= 2 ? 512 : 1024; }
#endif
constexpr int kEvalThreadsSmall = 256; // small launches (a few warps per SM): 255 registers per thread let ptxas schedule a round's lookups back to back

struct CmpAtomDev { uint64_t c; uint64_t root_off, cw_off, vb_off; int k; int pad; };
struct EvalArgs {
    const uint8_t *key[2]; const uint64_t *xhat;
    uint64_t *bits_out[2];      // [count] per slot, or null (call not wanted)
    uint64_t *coeff_out[2];     // [p][count] per slot, or null
    size_t count, s16, s8, lut_c, vt_first, vt_stride, lvl_stride, vt_lvl_rel, vt_fin_rel;
    uint64_t mask;
    int n, M, T, Gc, Gl, n_slots, party0, zero_first, et, pad;   // et: bit trees are early-terminated (variant bit 3, DESIGN 13)
    CmpAtomDev atom[kMaxAtoms];
};

__device__ __forceinline__ uint4 ld_stream16(const void *p) { return __ldcs(reinterpret_cast<const uint4 *>(p)); }
__device__ __forceinline__ uint64_t ld_stream8(const void *p) { return __ldcs(reinterpret_cast<const unsigned long long *>(p)); }

// (*p + v) mod 2^n for n < 64 without a fix-up pass: compare-and-swap loop (only used by small launches with G > 1)
__device__ __forceinline__ void atomic_add_ring(uint64_t *p, uint64_t v, uint64_t mask) {
    if (mask == ~0ull) { atomicAdd(reinterpret_cast<unsigned long long *>(p), (unsigned long long)v); return; }
    unsigned long long old = *reinterpret_cast<volatile unsigned long long *>(p), seen;
    do { seen = old; old = atomicCAS(reinterpret_cast<unsigned long long *>(p), seen, (seen + v) & mask); } while (old != seen);
}

// bit-DCF walk of one query; u = the k-bit public point, MSB-aligned.  With early termination (et) the tree has
// max(k-7, 0) levels and its leaf block holds the 2^min(k,7) output bits of the leaf's sub-range (DESIGN 13).
// STREAM: the key is read once (ld.global.cs); otherwise it is re-read for several points of the same element (ld.global.nc).
template <bool STREAM> __device__ __forceinline__ uint4 ld_key16(const void *p) {
    return STREAM ? __ldcs(reinterpret_cast<const uint4 *>(p)) : __ldg(reinterpret_cast<const uint4 *>(p));
}
template <bool STREAM> __device__ __forceinline__ uint64_t ld_key8(const void *p) {
    return STREAM ? __ldcs(reinterpret_cast<const unsigned long long *>(p)) : __ldg(reinterpret_cast<const unsigned long long *>(p));
}
template <bool STREAM>
__device__ __forceinline__ uint32_t bit_tree_eval(uint32_t tl, const uint8_t *key, size_t root_off, size_t cw_off, size_t vb_off,
                                                  size_t e, size_t s16, int k, uint64_t u, int party, int et) {
    uint4 s = ld_key16<STREAM>(key + root_off + e * 16);
    const uint64_t vb = ld_key8<STREAM>(key + vb_off + e * 8);
    const uint32_t fin = s.x & 1u;
    s.x &= ~3u;
    uint32_t tb = (uint32_t)party, V = 0;
    const int levels = et ? (k > 7 ? k - 7 : 0) : k;
    const uint8_t *cwp = key + cw_off + e * 16;
    uint4 cw = ld_key16<STREAM>(cwp);                                         // level 0, or (levels == 0) the leaf correction block
    for (int i = 0; i < levels; ++i) {
        uint4 cw_next = cw;
        if (i + 1 < levels + et) cw_next = ld_key16<STREAM>(cwp + (size_t)(i + 1) * s16);   // et: array `levels` = the 128-bit leaf CW
        const uint32_t dbit = (uint32_t)(u >> 63);
        u <<= 1;
        uint32_t x[1][4] = {{s.x | dbit, s.y, s.z, s.w}};
        uint32_t o[1][1][4];
        prg_blocks<1, 1, 0>(tl, x, o);
        const uint32_t tm = 0u - tb;                                          // all-ones iff the control bit is set
        V ^= ((o[0][0][0] >> 1) & 1u) ^ (tb & (uint32_t)((vb >> i) & 1ull));
        const uint32_t tnew = (o[0][0][0] & 1u) ^ (tb & (cw.x >> dbit) & 1u);
        s.x = (o[0][0][0] & ~3u) ^ (cw.x & ~3u & tm);
        s.y = o[0][0][1] ^ (cw.y & tm);
        s.z = o[0][0][2] ^ (cw.z & tm);
        s.w = o[0][0][3] ^ (cw.w & tm);
        tb = tnew;
        cw = cw_next;
    }
    uint32_t x[1][4] = {{s.x | 2u, s.y, s.z, s.w}};                           // leaf conversion, tweak 2
    uint32_t o[1][1][4];
    prg_blocks<1, 1, 0>(tl, x, o);
    if (!et) return (V ^ ((o[0][0][0] >> 1) & 1u) ^ (tb & fin)) & 1u;
    // leaf block = conv(s) ^ t * CW_leaf; bit (remaining input bits) of it; the level contributions V are scalar bits
    const uint32_t tm = 0u - tb;
    const uint32_t b0 = o[0][0][0] ^ (cw.x & tm), b1 = o[0][0][1] ^ (cw.y & tm), b2 = o[0][0][2] ^ (cw.z & tm), b3 = o[0][0][3] ^ (cw.w & tm);
    const int lowbits = k > 7 ? 7 : k;
    const uint32_t idx = (uint32_t)(u >> (64 - lowbits));                     // the remaining (low) input bits
    const uint32_t wsel = idx >> 5;
    const uint32_t word = wsel == 0 ? b0 : wsel == 1 ? b1 : wsel == 2 ? b2 : b3;
    return (V ^ (word >> (idx & 31u))) & 1u;
}

// the atoms t = g, g+G, .. of one element: packed XOR-share bits
__device__ __forceinline__ uint64_t cmp_item(const EvalArgs &a, uint32_t tl, const uint8_t *key, int party, size_t e, uint64_t xh, int g) {
    uint64_t word = 0;
    for (int t = g; t < a.T; t += a.Gc) {
        const CmpAtomDev &at = a.atom[t];
        const int k = at.k;
        const uint64_t km = k >= 64 ? ~0ull : ((1ull << k) - 1ull);
        const uint64_t u = (((xh & km) + at.c) & km) << (64 - k);             // view_{k,c}(xhat), MSB-aligned
        word |= (uint64_t)bit_tree_eval<true>(tl, key, at.root_off, at.cw_off, at.vb_off, e, a.s16, k, u, party, a.et) << t;
    }
    return word;
}

// the lookup trees j = 1+g, 1+g+G, .. of one element: acc += (-1)^party Eval(key_j, xhat); group 0 adds the constant share c_b
template <int P>
__device__ __forceinline__ void lut_item(const EvalArgs &a, uint32_t tl, const uint8_t *key, int party, size_t e, uint64_t xh_aligned, int g,
                                         uint64_t (&acc)[P]) {
    constexpr int Q = (P + 1) / 2;
#pragma unroll
    for (int w = 0; w < P; ++w) acc[w] = g == 0 ? ld_stream8(key + a.lut_c + (size_t)w * a.s8 + e * 8) : 0ull;
    for (int j = 1 + g; j < a.M; j += a.Gl) {
        const uint8_t *tree = key + a.vt_first + (size_t)(j - 1) * a.vt_stride;
        uint4 s = ld_stream16(tree + e * 16);
        s.x &= ~3u;
        uint32_t tb = (uint32_t)party;
        uint64_t V[P];
#pragma unroll
        for (int w = 0; w < P; ++w) V[w] = 0;
        const uint8_t *lvl = tree + a.vt_lvl_rel;
        uint64_t u = xh_aligned;
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
            acc[w] += party ? 0ull - v : v;
        }
    }
}

// grid-stride zeroing of the outputs that are accumulated with atomics, then one grid-wide barrier (cooperative launch)
__device__ __forceinline__ void zero_outputs_and_sync(uint64_t *const (&bits)[2], bool zero_bits, uint64_t *const (&coeff)[2], bool zero_coeff,
                                                      size_t count, int p) {
    const size_t tid = (size_t)blockIdx.x * blockDim.x + threadIdx.x, nth = (size_t)gridDim.x * blockDim.x;
    for (int s = 0; s < 2; ++s) {
        if (zero_bits && bits[s]) for (size_t i = tid; i < count; i += nth) bits[s][i] = 0;
        if (zero_coeff && coeff[s]) for (size_t i = tid; i < count * (size_t)p; i += nth) coeff[s][i] = 0;
    }
    __threadfence();
    cooperative_groups::this_grid().sync();
}

// THREADS = kEvalThreads (64 registers) or kEvalThreadsSmall (up to 255 registers: small launches run a few warps per SM and
// live on instruction-level parallelism inside each warp)
template <int P, int THREADS>
__global__ void __launch_bounds__(THREADS, 1) k_eval_p3(const __grid_constant__ EvalArgs a) {
    extern __shared__ uint32_t sT[];
    const uint32_t tl = aes_fill_tables(sT);
    if (a.zero_first) zero_outputs_and_sync(a.bits_out, a.Gc > 1, a.coeff_out, a.Gl > 1, a.count, P);
    const int lane = threadIdx.x & 31;
    const size_t tiles = (a.count + 31) / 32;
    const bool any_lut = a.M > 1 && (a.coeff_out[0] || a.coeff_out[1]), any_cmp = a.T > 0 && (a.bits_out[0] || a.bits_out[1]);
    const size_t lut_per_slot = any_lut ? tiles * (size_t)a.Gl : 0, cmp_per_slot = any_cmp ? tiles * (size_t)a.Gc : 0;
    const size_t n_lut = lut_per_slot * (size_t)a.n_slots, items = n_lut + cmp_per_slot * (size_t)a.n_slots;
    const size_t warps = (size_t)gridDim.x * (blockDim.x >> 5);
    // warp w of CTA b takes the items w*grid + b (+ k*warps): a partial last wave spreads over all SMs; the long (lookup) items come first
    for (size_t it = (size_t)(threadIdx.x >> 5) * gridDim.x + blockIdx.x; it < items; it += warps) {
        const bool is_lut = it < n_lut;
        const size_t r = is_lut ? it : it - n_lut, per_slot = is_lut ? lut_per_slot : cmp_per_slot;
        const int slot = (int)(r / per_slot);
        const size_t r2 = r - (size_t)slot * per_slot;
        const int g = (int)(r2 / tiles);
        const size_t tile = r2 - (size_t)g * tiles;
        const int party = a.n_slots == 2 ? slot : a.party0;
        const uint8_t *key = a.key[slot];
        size_t e = tile * 32 + lane;
        const bool live = e < a.count;
        if (!live) e = a.count - 1;
        const uint64_t xh = a.xhat[e];
        if (is_lut) {
            if (!a.coeff_out[slot]) continue;
            uint64_t acc[P];
            lut_item<P>(a, tl, key, party, e, (xh & a.mask) << (64 - a.n), g, acc);
            if (live) {
#pragma unroll
                for (int w = 0; w < P; ++w) {
                    uint64_t *dst = a.coeff_out[slot] + (size_t)w * a.count + e;
                    if (a.Gl == 1) *dst = acc[w] & a.mask;
                    else atomic_add_ring(dst, acc[w] & a.mask, a.mask);
                }
            }
        } else {
            if (!a.bits_out[slot]) continue;
            const uint64_t word = cmp_item(a, tl, key, party, e, xh, g);
            if (live) {
                if (a.Gc == 1) a.bits_out[slot][e] = word;
                else atomicOr(reinterpret_cast<unsigned long long *>(a.bits_out[slot] + e), (unsigned long long)word);
            }
        }
    }
}

}  // namespace fsk
