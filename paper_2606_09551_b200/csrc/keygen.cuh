// keygen.cuh -- dealer kernels (section 5.2): per element, T bit-DCF Gen (a2), Protocol 3 step (1)
// + (M-1) vector-DCF Gen + additive split of v_{M-1} (a1, a3), and the share splitting of masks,
// instance constants and correlated randomness (a4).  DCF Gen: DESIGN 4.2; randomness slots: DESIGN 4.5;
// key layout: DESIGN 4.4.  One lane per element, one warp per (32-element tile, tree): the level loop is
// sequential, the four child expansions of a level run in lock-step through the shared-memory T-tables, and
// each level's correction words are written to both parties' buffers as coalesced streaming stores.
#pragma once
#include "aes.cuh"

namespace fsk {

constexpr int kGenThreads = 512;

enum : uint64_t {
    SLOT_BIT_ROOT = 0x1000, SLOT_VEC_ROOT = 0x2000, SLOT_LUT_C = 0x3000, SLOT_RIN = 0x4000, SLOT_ROUT = 0x4100,
    SLOT_KA = 0x5000, SLOT_KB = 0x5800, SLOT_BV_AB = 0x6000, SLOT_BV_AB0 = 0x6800, SLOT_BV_C0 = 0x7000,
    SLOT_AND_AB = 0x8000, SLOT_AND_AB0 = 0x8001, SLOT_AND_C0 = 0x8002, SLOT_B2A = 0x9000, SLOT_B2A_A0 = 0x9100,
    SLOT_A2B_RHO = 0xB000, SLOT_A2B_RHO0 = 0xB100, SLOT_A2B_BITS = 0xB200       // A2B (DESIGN 15); its tree roots: 0x1800 + 2i + b
};

__device__ __forceinline__ void st_stream16(void *p, uint4 v) { __stcs(reinterpret_cast<uint4 *>(p), v); }
__device__ __forceinline__ void st_stream8(void *p, uint64_t v) { __stcs(reinterpret_cast<unsigned long long *>(p), (unsigned long long)v); }

// R(e, slot) = AES_{seed||~seed}(LE64(e) || LE64(slot))
__device__ __forceinline__ void dealer_rand(uint32_t tl, const RoundKeys &rk, uint64_t e, uint64_t slot, uint64_t &lo, uint64_t &hi) {
    uint32_t s[4] = {(uint32_t)e, (uint32_t)(e >> 32), (uint32_t)slot, (uint32_t)(slot >> 32)};
    aes_encrypt_rk(tl, rk, s);
    lo = (uint64_t)s[0] | ((uint64_t)s[1] << 32);
    hi = (uint64_t)s[2] | ((uint64_t)s[3] << 32);
}

// is_theta: 0 = r-atom (threshold r_k), 1 = theta-atom (r_k + beta), 2 = A2B key i (threshold rho_i mod 2^k, rho_i = R(e, 0xB000 + i))
struct GenAtomDev { uint64_t c, beta, root_off, cw_off, vb_off; int k, is_theta; };
struct GenBitArgs {
    uint8_t *key0, *key1; const uint64_t *r_in;
    size_t count, s16; uint64_t first_elem, mask;
    int T, et;                 // et: early-terminated trees (variant bit 3, DESIGN 13): max(k-7,0) levels + a 128-bit leaf block
    int slot_t0, pad;          // tree t draws its roots from R(e, 0x1000 + 2 (slot_t0 + t) + b): 0 for the atoms, 0x400 for the A2B keys
    RoundKeys rk;
    GenAtomDev atom[kMaxAtoms];
};

// the body of k_gen_bit (also run by k_gen_tiny, which makes ONE launch of a tiny tensor's whole dealer step)
__device__ __forceinline__ void gen_bit_body(const GenBitArgs &a, const uint32_t tl) {
    const int lane = threadIdx.x & 31;
    const size_t tiles = (a.count + 31) / 32;
    const size_t items = tiles * (size_t)a.T;
    const size_t warps = (size_t)gridDim.x * (blockDim.x >> 5);
    for (size_t it = (size_t)(threadIdx.x >> 5) * gridDim.x + blockIdx.x; it < items; it += warps) {   // warp w of CTA b takes items w*grid + b: a partial last wave spreads over all SMs
        const int t = (int)(it / tiles);
        const size_t e = (it - (size_t)t * tiles) * 32 + lane;
        if (e >= a.count) continue;
        const GenAtomDev &at = a.atom[t];
        const int k = at.k;
        if (k == 0) continue;                              // variant 1: slot of the n-bit view (its key is a vector tree)
        const uint64_t km = k >= 64 ? ~0ull : ((1ull << k) - 1ull);
        uint64_t rk_ = a.r_in[e] & a.mask & km;
        if (at.is_theta == 2) {                            // A2B key t: the threshold is the low k bits of the dealer's mask rho_t
            uint64_t lo, hi;
            dealer_rand(tl, a.rk, a.first_elem + e, SLOT_A2B_RHO + t, lo, hi);
            rk_ = lo & a.mask & km;
        }
        // threshold of the masked comparison (Lemma 4.3 / E.1): theta = (r_k + beta) mod 2^k, or r_k for the r-atom
        uint64_t alpha = (at.is_theta == 1 ? (rk_ + at.beta) & km : rk_) << (64 - k);
        uint32_t s[2][4];
        {
            uint64_t lo, hi;
            dealer_rand(tl, a.rk, a.first_elem + e, SLOT_BIT_ROOT + 2 * (a.slot_t0 + t), lo, hi);
            s[0][0] = (uint32_t)lo & ~3u; s[0][1] = (uint32_t)(lo >> 32); s[0][2] = (uint32_t)hi; s[0][3] = (uint32_t)(hi >> 32);
            dealer_rand(tl, a.rk, a.first_elem + e, SLOT_BIT_ROOT + 2 * (a.slot_t0 + t) + 1, lo, hi);
            s[1][0] = (uint32_t)lo & ~3u; s[1][1] = (uint32_t)(lo >> 32); s[1][2] = (uint32_t)hi; s[1][3] = (uint32_t)(hi >> 32);
        }
        const uint4 root0 = make_uint4(s[0][0], s[0][1], s[0][2], s[0][3]);
        const uint4 root1 = make_uint4(s[1][0], s[1][1], s[1][2], s[1][3]);
        uint32_t t0 = 0, t1 = 1, Va = 0;
        uint64_t vbits = 0;
        uint8_t *cw0 = a.key0 + at.cw_off + e * 16, *cw1 = a.key1 + at.cw_off + e * 16;
        const int levels = a.et ? (k > 7 ? k - 7 : 0) : k;             // the tree walks the top `levels` bits of alpha
        for (int i = 0; i < levels; ++i) {
            const uint32_t abit = (uint32_t)(alpha >> 63);
            alpha <<= 1;
            // children: index 2*b + d
            uint32_t o[4][1][4];
#pragma unroll
            for (int b = 0; b < 2; ++b) {
                uint32_t x[2][4], ob[2][1][4];
#pragma unroll
                for (int d = 0; d < 2; ++d) { x[d][0] = s[b][0] | (uint32_t)d; x[d][1] = s[b][1]; x[d][2] = s[b][2]; x[d][3] = s[b][3]; }
                prg_blocks<2, 1, 0, true, 3>(tl, x, ob);
#pragma unroll
                for (int d = 0; d < 2; ++d)
#pragma unroll
                    for (int c = 0; c < 4; ++c) o[2 * b + d][0][c] = ob[d][0][c];
            }
            const uint32_t am = 0u - abit;                    // keep = alpha_i, lose = 1 - alpha_i
            uint32_t keep0[4], keep1[4], scw[4];
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                const uint32_t l0 = (o[1][0][c] & ~am) | (o[0][0][c] & am);       // lose = 1 when abit = 0
                const uint32_t l1 = (o[3][0][c] & ~am) | (o[2][0][c] & am);
                keep0[c] = (o[0][0][c] & ~am) | (o[1][0][c] & am);
                keep1[c] = (o[2][0][c] & ~am) | (o[3][0][c] & am);
                scw[c] = l0 ^ l1;
            }
            // word 0 carries: bit0 = control bit T, bit1 = Z_2 payload W
            const uint32_t lose_w = ((scw[0] >> 1) & 1u);                          // W_0[lose] ^ W_1[lose]
            const uint32_t keep_w = ((keep0[0] ^ keep1[0]) >> 1) & 1u;
            const uint32_t vcw = lose_w ^ Va ^ (abit);                             // + beta (=1) iff lose = 0 iff alpha_i = 1
            Va ^= keep_w ^ vcw;
            const uint32_t tcw0 = ((o[0][0][0] ^ o[2][0][0]) & 1u) ^ abit ^ 1u;
            const uint32_t tcw1 = ((o[1][0][0] ^ o[3][0][0]) & 1u) ^ abit;
            const uint32_t tcw_keep = abit ? tcw1 : tcw0;
            scw[0] = (scw[0] & ~3u) | tcw0 | (tcw1 << 1);
            const uint4 cwv = make_uint4(scw[0], scw[1], scw[2], scw[3]);
            st_stream16(cw0 + (size_t)i * a.s16, cwv);
            st_stream16(cw1 + (size_t)i * a.s16, cwv);
            vbits |= (uint64_t)vcw << i;
            const uint32_t m0 = 0u - t0, m1 = 0u - t1;
            const uint32_t nt0 = (keep0[0] & 1u) ^ (t0 & tcw_keep), nt1 = (keep1[0] & 1u) ^ (t1 & tcw_keep);
            s[0][0] = (keep0[0] & ~3u) ^ (scw[0] & ~3u & m0); s[1][0] = (keep1[0] & ~3u) ^ (scw[0] & ~3u & m1);
#pragma unroll
            for (int c = 1; c < 4; ++c) { s[0][c] = keep0[c] ^ (scw[c] & m0); s[1][c] = keep1[c] ^ (scw[c] & m1); }
            t0 = nt0; t1 = nt1;
        }
        uint32_t x[2][4], o[2][1][4];
#pragma unroll
        for (int b = 0; b < 2; ++b) { x[b][0] = s[b][0] | 2u; x[b][1] = s[b][1]; x[b][2] = s[b][2]; x[b][3] = s[b][3]; }
        prg_blocks<2, 1, 0>(tl, x, o);
        uint32_t fin = (((o[0][0][0] ^ o[1][0][0]) >> 1) & 1u) ^ Va;
        if (a.et) {
            // leaf correction block L = conv128(s_0) ^ conv128(s_1) ^ X, X_j = Valpha ^ I[j < alpha_lo], alpha_lo = the remaining low bits
            const int lam = k - levels;
            const uint32_t alo = (uint32_t)(alpha >> (64 - lam));
            const uint32_t vm = 0u - Va;
            uint32_t L[4];
#pragma unroll
            for (int w = 0; w < 4; ++w) {
                const uint32_t below = alo >= 32u * (w + 1) ? ~0u : alo <= 32u * w ? 0u : ((1u << (alo - 32u * w)) - 1u);
                L[w] = o[0][0][w] ^ o[1][0][w] ^ below ^ vm;
            }
            const uint4 lv = make_uint4(L[0], L[1], L[2], L[3]);
            st_stream16(cw0 + (size_t)levels * a.s16, lv);
            st_stream16(cw1 + (size_t)levels * a.s16, lv);
            fin = 0;
        }
        st_stream16(a.key0 + at.root_off + e * 16, make_uint4(root0.x | fin, root0.y, root0.z, root0.w));
        st_stream16(a.key1 + at.root_off + e * 16, make_uint4(root1.x | fin, root1.y, root1.z, root1.w));
        st_stream8(a.key0 + at.vb_off + e * 8, vbits);
        st_stream8(a.key1 + at.vb_off + e * 8, vbits);
    }
}

__global__ void __launch_bounds__(kGenThreads, 1) k_gen_bit(const __grid_constant__ GenBitArgs a) {
    extern __shared__ uint32_t sT[];
    gen_bit_body(a, aes_fill_tables(sT));
}


// ---------------------------------------------------------------------------------------------------
// Protocol 3 step (1) for one element, evaluated per lookup interval j on demand.
// The sort of s_i = (alpha_i + r) mod N is always the cyclic rotation pi(q) = (i0 + q) mod m with
// i0 = #{i : alpha_i + r < N} (the non-wrapping starts stay in order and follow the wrapped ones).
// ---------------------------------------------------------------------------------------------------
struct P3 {
    const uint64_t *alpha;     // interior boundaries alpha_1..alpha_{m-1}
    uint64_t r, mask, N;       // N = 2^n (0 when n = 64: differences are taken mod 2^64)
    int m, n, i0, beta0_zero, jstar;
    __device__ __forceinline__ uint64_t start(int i) const { return ((i == 0 ? 0ull : alpha[i - 1]) + r) & mask; }
    __device__ __forceinline__ int pi(int q) const { int v = i0 + q; return v >= m ? v - m : v; }
    __device__ __forceinline__ uint64_t sorted(int q) const { return start(pi(q)); }          // beta_q
    __device__ void init(const uint64_t *alpha_, int m_, int n_, uint64_t mask_, uint64_t r_, int M) {
        alpha = alpha_; m = m_; n = n_; mask = mask_; r = r_; N = n_ >= 64 ? 0ull : (1ull << n_);
        i0 = 0;
        for (int i = 0; i < m; ++i) {
            const uint64_t a_i = i == 0 ? 0ull : alpha[i - 1];
            const uint64_t sum = a_i + r;
            const bool wraps = n >= 64 ? sum < a_i : (sum >> n) != 0;
            i0 += wraps ? 0 : 1;
        }
        beta0_zero = sorted(0) == 0;
        jstar = -1;
        if (beta0_zero && M == m + 1) {                                  // lines 12-18: dummy split at the first gap >= 2
            for (int j = 0; j < m && jstar < 0; ++j) {
                const uint64_t lo = sorted(j);                           // B'_j  (B'_0 = beta_0 = 0)
                const uint64_t hi = j + 1 == m ? N : sorted(j + 1);      // B'_m = N (0 mod 2^64 when n = 64; lo >= 1 there)
                if (hi - lo >= 2) jstar = j;
            }
        }
    }
    // boundary B_q (1 <= q <= M-1) and interval label ord_q (0 <= q <= M-1)
    __device__ __forceinline__ uint64_t B(int q) const {
        if (!beta0_zero) return sorted(q - 1);                           // line 19: B = (0, beta_0, .., beta_{m-1}, N)
        if (jstar < 0 || q <= jstar) return sorted(q);
        if (q == jstar + 1) return sorted(jstar) + 1;                    // delta = B_{j*} + 1
        return sorted(q - 1);
    }
    __device__ __forceinline__ int ord(int q) const {
        if (!beta0_zero) return q == 0 ? pi(m - 1) : pi(q - 1);
        if (jstar < 0 || q <= jstar) return pi(q);
        return pi(q - 1);
    }
};

// variant bit 2 (DESIGN 11): replace the coefficients of every polynomial of a payload (high degree first, d+1 words
// each, `polys` of them) by those of P(X - r): Taylor shift by synthetic division, d passes of c_idx += (-r) c_{idx-1}.
template <int P>
__device__ __forceinline__ void shift_payload(uint64_t (&v)[P], int polys, int d, uint64_t negr) {
    const int nc = polys * (d + 1);
    for (int it = 0; it < d; ++it) {
#pragma unroll
        for (int w = 1; w < P; ++w) {
            const int idx = w % (d + 1);
            if (w < nc && idx >= 1 && idx <= d - it) v[w] += negr * v[w - 1];
        }
    }
}

struct GenVecArgs {
    uint8_t *key0, *key1; const uint64_t *r_in; const uint64_t *alpha; const uint64_t *payload;   // payload[m][p]
    size_t count, s16, s8, vt_first, vt_stride, lvl_stride, vt_lvl_rel, vt_fin_rel;
    uint64_t first_elem, mask;
    int n, m, M, sp;           // sp = 1 (variant 1): the single tree f_{r,beta}: threshold r_in, beta = (1, -r, (-r)^2, ..), no Protocol 3
    int xpoly, polys, d, pad2; // variant bit 2 with Protocol 3: payloads are the coefficients of P_i(X - r_in)
    RoundKeys rk;
};

template <int P>
__global__ void __launch_bounds__(kGenThreads, 1) k_gen_vec(const __grid_constant__ GenVecArgs a) {
    constexpr int Q = (P + 1) / 2;
    extern __shared__ uint32_t sT[];
    const uint32_t tl = aes_fill_tables(sT);
    const int lane = threadIdx.x & 31;
    const size_t tiles = (a.count + 31) / 32;
    const size_t items = tiles * (size_t)(a.M - 1);
    const size_t warps = (size_t)gridDim.x * (blockDim.x >> 5);
    for (size_t it = (size_t)(threadIdx.x >> 5) * gridDim.x + blockIdx.x; it < items; it += warps) {   // warp w of CTA b takes items w*grid + b: a partial last wave spreads over all SMs
        const int j = 1 + (int)(it / tiles);
        const size_t e = (it - (size_t)(j - 1) * tiles) * 32 + lane;
        if (e >= a.count) continue;
        const uint64_t r = a.r_in[e] & a.mask;
        uint64_t alpha, beta[P];
        if (a.sp) {
            alpha = r << (64 - a.n);
            beta[0] = 1;
#pragma unroll
            for (int w = 1; w < P; ++w) beta[w] = beta[w - 1] * (0ull - r);
        } else {
            P3 p3;
            p3.init(a.alpha, a.m, a.n, a.mask, r, a.M);
            alpha = p3.B(j) << (64 - a.n);
            const uint64_t *va = a.payload + (size_t)p3.ord(j - 1) * P, *vb = a.payload + (size_t)p3.ord(j) * P;
#pragma unroll
            for (int w = 0; w < P; ++w) beta[w] = va[w] - vb[w];                // Delta_j = v_{j-1} - v_j
            if (a.xpoly) shift_payload<P>(beta, a.polys, a.d, 0ull - r);        // the shift is linear: shift the difference
        }
        uint32_t s[2][4];
        {
            uint64_t lo, hi;
            dealer_rand(tl, a.rk, a.first_elem + e, SLOT_VEC_ROOT + 2 * j, lo, hi);
            s[0][0] = (uint32_t)lo & ~3u; s[0][1] = (uint32_t)(lo >> 32); s[0][2] = (uint32_t)hi; s[0][3] = (uint32_t)(hi >> 32);
            dealer_rand(tl, a.rk, a.first_elem + e, SLOT_VEC_ROOT + 2 * j + 1, lo, hi);
            s[1][0] = (uint32_t)lo & ~3u; s[1][1] = (uint32_t)(lo >> 32); s[1][2] = (uint32_t)hi; s[1][3] = (uint32_t)(hi >> 32);
        }
        uint8_t *tree0 = a.key0 + a.vt_first + (size_t)(j - 1) * a.vt_stride;
        uint8_t *tree1 = a.key1 + a.vt_first + (size_t)(j - 1) * a.vt_stride;
        st_stream16(tree0 + e * 16, make_uint4(s[0][0], s[0][1], s[0][2], s[0][3]));
        st_stream16(tree1 + e * 16, make_uint4(s[1][0], s[1][1], s[1][2], s[1][3]));
        uint32_t t0 = 0, t1 = 1;
        uint64_t Va[P];
#pragma unroll
        for (int w = 0; w < P; ++w) Va[w] = 0;
        size_t lvl = a.vt_lvl_rel;
        for (int i = 0; i < a.n; ++i, lvl += a.lvl_stride) {
            const uint32_t abit = (uint32_t)(alpha >> 63);
            alpha <<= 1;
            const uint32_t am = 0u - abit;
            const uint64_t am64 = 0ull - (uint64_t)abit;
            uint32_t keepS[2][4], loseS[2][4], Tb[2][2];
            uint64_t keepW[2][P], loseW[2][P];
#pragma unroll
            for (int b = 0; b < 2; ++b) {                                  // party b: both directions in lock-step
                uint32_t x[2][4], o[2][1 + Q][4];
#pragma unroll
                for (int d = 0; d < 2; ++d) { x[d][0] = s[b][0] | (uint32_t)d; x[d][1] = s[b][1]; x[d][2] = s[b][2]; x[d][3] = s[b][3]; }
                prg_blocks<2, 1 + Q, 0, true>(tl, x, o);
                Tb[b][0] = o[0][0][0] & 1u; Tb[b][1] = o[1][0][0] & 1u;
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    const uint32_t v0 = c == 0 ? o[0][0][0] & ~3u : o[0][0][c], v1 = c == 0 ? o[1][0][0] & ~3u : o[1][0][c];
                    keepS[b][c] = (v0 & ~am) | (v1 & am);
                    loseS[b][c] = (v1 & ~am) | (v0 & am);
                }
#pragma unroll
                for (int w = 0; w < P; ++w) {
                    const uint64_t w0 = (uint64_t)o[0][1 + w / 2][2 * (w & 1)] | ((uint64_t)o[0][1 + w / 2][2 * (w & 1) + 1] << 32);
                    const uint64_t w1 = (uint64_t)o[1][1 + w / 2][2 * (w & 1)] | ((uint64_t)o[1][1 + w / 2][2 * (w & 1) + 1] << 32);
                    keepW[b][w] = (w0 & ~am64) | (w1 & am64);
                    loseW[b][w] = (w1 & ~am64) | (w0 & am64);
                }
            }
            uint32_t scw[4];
#pragma unroll
            for (int c = 0; c < 4; ++c) scw[c] = loseS[0][c] ^ loseS[1][c];
            const uint64_t sgn = 0ull - (uint64_t)t1;                       // (-1)^{t_1}: negate iff t_1 = 1
            uint64_t vcw[P];
#pragma unroll
            for (int w = 0; w < P; ++w) {
                uint64_t v = loseW[1][w] - loseW[0][w] - Va[w] + (beta[w] & am64);     // + beta iff lose = 0 iff alpha_i = 1
                v = ((v ^ sgn) - sgn) & a.mask;
                vcw[w] = v;
                Va[w] = Va[w] - keepW[1][w] + keepW[0][w] + ((v ^ sgn) - sgn);
            }
            const uint32_t tcw0 = Tb[0][0] ^ Tb[1][0] ^ abit ^ 1u, tcw1 = Tb[0][1] ^ Tb[1][1] ^ abit;
            const uint32_t tcw_keep = abit ? tcw1 : tcw0;
            const uint4 cwv = make_uint4(scw[0] | tcw0 | (tcw1 << 1), scw[1], scw[2], scw[3]);
            st_stream16(tree0 + lvl + e * 16, cwv);
            st_stream16(tree1 + lvl + e * 16, cwv);
#pragma unroll
            for (int w = 0; w < P; ++w) {
                st_stream8(tree0 + lvl + a.s16 + (size_t)w * a.s8 + e * 8, vcw[w]);
                st_stream8(tree1 + lvl + a.s16 + (size_t)w * a.s8 + e * 8, vcw[w]);
            }
            const uint32_t m0 = 0u - t0, m1 = 0u - t1;
            const uint32_t nt0 = (abit ? Tb[0][1] : Tb[0][0]) ^ (t0 & tcw_keep), nt1 = (abit ? Tb[1][1] : Tb[1][0]) ^ (t1 & tcw_keep);
#pragma unroll
            for (int c = 0; c < 4; ++c) { s[0][c] = keepS[0][c] ^ (scw[c] & m0); s[1][c] = keepS[1][c] ^ (scw[c] & m1); }
            t0 = nt0; t1 = nt1;
        }
        // final correction word: fin = (-1)^{t_1} (conv(s_1) - conv(s_0) - Valpha)
        uint32_t o[2][Q][4];
#pragma unroll
        for (int b = 0; b < 2; ++b) {
            uint32_t x[1][4] = {{s[b][0] | 2u, s[b][1], s[b][2], s[b][3]}}, ob[1][Q][4];
            prg_blocks<1, Q, 1, true>(tl, x, ob);
#pragma unroll
            for (int q = 0; q < Q; ++q)
#pragma unroll
                for (int c = 0; c < 4; ++c) o[b][q][c] = ob[0][q][c];
        }
        const uint64_t sgn = 0ull - (uint64_t)t1;
#pragma unroll
        for (int w = 0; w < P; ++w) {
            const uint64_t c0 = (uint64_t)o[0][w / 2][2 * (w & 1)] | ((uint64_t)o[0][w / 2][2 * (w & 1) + 1] << 32);
            const uint64_t c1 = (uint64_t)o[1][w / 2][2 * (w & 1)] | ((uint64_t)o[1][w / 2][2 * (w & 1) + 1] << 32);
            uint64_t v = c1 - c0 - Va[w];
            v = ((v ^ sgn) - sgn) & a.mask;
            st_stream8(tree0 + a.vt_fin_rel + (size_t)w * a.s8 + e * 8, v);
            st_stream8(tree1 + a.vt_fin_rel + (size_t)w * a.s8 + e * 8, v);
        }
    }
}


// ---------------------------------------------------------------------------------------------------
// k_gen_vec for SMALL launches (a few thousand elements: relu16, recip, rsqrt).  There the machine is far from full and what
// bounds the dealer is the chain of one tree: n levels x the 4 (1+Q) PRG blocks a lane of k_gen_vec expands per level.  Here a
// QUAD of lanes shares one element: lane 4 q + c expands child c = 2 b + d (party b, direction d) only, so a level's critical path
// is 1+Q blocks, and the correction words are assembled with warp shuffles (about 35 per level).  A warp = (8-element tile, tree).
// Same arithmetic, same bytes: every value below is the one k_gen_vec computes (DESIGN 4.2), only WHERE it is computed differs.
// ---------------------------------------------------------------------------------------------------
template <int P>
__device__ __forceinline__ void gen_vec_quad_body(const GenVecArgs &a, const uint32_t tl) {
    constexpr int Q = (P + 1) / 2;
    constexpr unsigned FULL = 0xffffffffu;
    const int lane = threadIdx.x & 31, c = lane & 3, b = c >> 1, d = c & 1, base = lane & ~3;
    const size_t tiles = (a.count + 7) / 8;
    const size_t items = tiles * (size_t)(a.M - 1);
    const size_t warps = (size_t)gridDim.x * (blockDim.x >> 5);
    for (size_t it = (size_t)(threadIdx.x >> 5) * gridDim.x + blockIdx.x; it < items; it += warps) {
        const int j = 1 + (int)(it / tiles);
        size_t e = (it - (size_t)(j - 1) * tiles) * 8 + (size_t)(lane >> 2);
        const bool live = e < a.count;                                   // dead quads shadow the last element and store nothing
        if (!live) e = a.count - 1;
        const uint64_t r = a.r_in[e] & a.mask;
        uint64_t alpha, beta[P];
        if (a.sp) {
            alpha = r << (64 - a.n);
            beta[0] = 1;
#pragma unroll
            for (int w = 1; w < P; ++w) beta[w] = beta[w - 1] * (0ull - r);
        } else {
            P3 p3;
            p3.init(a.alpha, a.m, a.n, a.mask, r, a.M);
            alpha = p3.B(j) << (64 - a.n);
            const uint64_t *va = a.payload + (size_t)p3.ord(j - 1) * P, *vb = a.payload + (size_t)p3.ord(j) * P;
#pragma unroll
            for (int w = 0; w < P; ++w) beta[w] = va[w] - vb[w];
            if (a.xpoly) shift_payload<P>(beta, a.polys, a.d, 0ull - r);
        }
        uint32_t s[4];                                                   // this lane's party's seed
        {
            uint64_t lo, hi;
            dealer_rand(tl, a.rk, a.first_elem + e, SLOT_VEC_ROOT + 2 * j + b, lo, hi);
            s[0] = (uint32_t)lo & ~3u; s[1] = (uint32_t)(lo >> 32); s[2] = (uint32_t)hi; s[3] = (uint32_t)(hi >> 32);
        }
        uint8_t *tree0 = a.key0 + a.vt_first + (size_t)(j - 1) * a.vt_stride;
        uint8_t *tree1 = a.key1 + a.vt_first + (size_t)(j - 1) * a.vt_stride;
        uint8_t *mytree = (c & 1) ? tree1 : tree0;                       // lanes 0 / 1 store the seed words, lanes 2 / 3 the payload words
        if (live && d == 0) st_stream16((b ? tree1 : tree0) + e * 16, make_uint4(s[0], s[1], s[2], s[3]));
        uint32_t t0 = 0, t1 = 1;                                         // replicated in the four lanes
        uint64_t Va[P];
#pragma unroll
        for (int w = 0; w < P; ++w) Va[w] = 0;
        size_t lvl = a.vt_lvl_rel;
        for (int i = 0; i < a.n; ++i, lvl += a.lvl_stride) {
            const uint32_t abit = (uint32_t)(alpha >> 63);
            alpha <<= 1;
            const uint64_t am64 = 0ull - (uint64_t)abit;
            const int keep_d = (int)abit, lose_d = 1 - keep_d;
            uint32_t x[1][4] = {{s[0] | (uint32_t)d, s[1], s[2], s[3]}}, o[1][1 + Q][4];
            prg_blocks<1, 1 + Q, 0, 1>(tl, x, o);
            const uint32_t T = o[0][0][0] & 1u;
            uint32_t S[4] = {o[0][0][0] & ~3u, o[0][0][1], o[0][0][2], o[0][0][3]};
            uint32_t scw[4], keepS[4];
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const uint32_t sx = S[k] ^ __shfl_xor_sync(FULL, S[k], 2);           // S_0[d] ^ S_1[d]
                scw[k] = __shfl_sync(FULL, sx, base + lose_d);
                keepS[k] = __shfl_sync(FULL, S[k], base + 2 * b + keep_d);            // S_b[keep]
            }
            const uint32_t tx = T ^ __shfl_xor_sync(FULL, T, 2);                      // T_0[d] ^ T_1[d]
            const uint32_t tcw0 = __shfl_sync(FULL, tx, base) ^ abit ^ 1u, tcw1 = __shfl_sync(FULL, tx, base + 1) ^ abit;
            const uint32_t tcw_keep = abit ? tcw1 : tcw0;
            const uint32_t Tk0 = __shfl_sync(FULL, T, base + keep_d), Tk1 = __shfl_sync(FULL, T, base + 2 + keep_d);
            const uint64_t sgn = 0ull - (uint64_t)t1;
            uint64_t vcw[P];
#pragma unroll
            for (int w = 0; w < P; ++w) {
                const uint64_t W = (uint64_t)o[0][1 + w / 2][2 * (w & 1)] | ((uint64_t)o[0][1 + w / 2][2 * (w & 1) + 1] << 32);
                const uint64_t Wp = __shfl_xor_sync(FULL, W, 2);
                const uint64_t D = b ? W - Wp : Wp - W;                                // W_1[d] - W_0[d]
                const uint64_t loseD = __shfl_sync(FULL, D, base + lose_d), keepD = __shfl_sync(FULL, D, base + keep_d);
                uint64_t v = loseD - Va[w] + (beta[w] & am64);
                v = ((v ^ sgn) - sgn) & a.mask;
                vcw[w] = v;
                Va[w] = Va[w] - keepD + ((v ^ sgn) - sgn);
            }
            if (live) {
                if (c < 2) st_stream16(mytree + lvl + e * 16, make_uint4(scw[0] | tcw0 | (tcw1 << 1), scw[1], scw[2], scw[3]));
                else {
#pragma unroll
                    for (int w = 0; w < P; ++w) st_stream8(mytree + lvl + a.s16 + (size_t)w * a.s8 + e * 8, vcw[w]);
                }
            }
            const uint32_t tb = b ? t1 : t0, mb = 0u - tb;
#pragma unroll
            for (int k = 0; k < 4; ++k) s[k] = keepS[k] ^ (scw[k] & mb);
            const uint32_t nt0 = Tk0 ^ (t0 & tcw_keep), nt1 = Tk1 ^ (t1 & tcw_keep);
            t0 = nt0; t1 = nt1;
        }
        // final correction word: fin = (-1)^{t_1} (conv(s_1) - conv(s_0) - Valpha)
        uint32_t x[1][4] = {{s[0] | 2u, s[1], s[2], s[3]}}, o[1][Q][4];
        prg_blocks<1, Q, 1, 1>(tl, x, o);
        const uint64_t sgn = 0ull - (uint64_t)t1;
#pragma unroll
        for (int w = 0; w < P; ++w) {
            const uint64_t C = (uint64_t)o[0][w / 2][2 * (w & 1)] | ((uint64_t)o[0][w / 2][2 * (w & 1) + 1] << 32);
            const uint64_t Cp = __shfl_xor_sync(FULL, C, 2);
            uint64_t v = (b ? C - Cp : Cp - C) - Va[w];
            v = ((v ^ sgn) - sgn) & a.mask;
            if (live && c < 2) st_stream8(mytree + a.vt_fin_rel + (size_t)w * a.s8 + e * 8, v);
        }
    }
}

template <int P>
__global__ void __launch_bounds__(kGenThreads, 1) k_gen_vec_quad(const __grid_constant__ GenVecArgs a) {
    extern __shared__ uint32_t sT[];
    gen_vec_quad_body<P>(a, aes_fill_tables(sT));
}


// ---------------------------------------------------------------------------------------------------
// a4: share splitting.  One lane per element: c_b of the lookup, [r_in], [r_out], kappa^A,
// kappa^B (theta-atom carries of Lemma 4.3 + the spec's bits), Beaver / AND / B2A material.
// ---------------------------------------------------------------------------------------------------
struct GenMiscArgs {
    uint8_t *key0, *key1; const uint64_t *r_in, *r_out, *alpha, *payload;
    size_t count, s8, lut_c, rin, rout, ka, kb, beaver, andt, b2a_bits, b2a_a, rpow, a2b_rho, a2b_bits;
    int xpoly, polys, d, n_rpow;
    int GA2B, a2b_bit[kMaxA2B], pad3;
    uint64_t first_elem, mask;
    int n, m, M, p, has_lut, mask_output, n_out_a, n_ka, n_kb_spec, n_carry, T, MA, MB, GMIX;
    uint64_t ma_is_x;          // bit i: arithmetic gate i is a product with the gate input (material (b, c = b r_in), DESIGN 10)
    RoundKeys rk;
    uint8_t ka_kind[8], ka_arg[8], kb_kind[64], kb_arg[64];
    GenAtomDev atom[kMaxAtoms];
};

__device__ __forceinline__ void gen_misc_body(const GenMiscArgs &a, const uint32_t tl) {
    for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < a.count; e += (size_t)gridDim.x * blockDim.x) {
        const uint64_t ge = a.first_elem + e;
        const uint64_t r = a.r_in[e] & a.mask;
        uint64_t lo, hi;
        auto put = [&](size_t off, uint64_t v0, uint64_t v1) {
            st_stream8(a.key0 + off + e * 8, v0);
            st_stream8(a.key1 + off + e * 8, v1);
        };
        if (a.has_lut) {                                                   // additive split of v_{M-1}
            P3 p3;
            p3.init(a.alpha, a.m, a.n, a.mask, r, a.M);
            const uint64_t *vp = a.payload + (size_t)p3.ord(a.M - 1) * a.p;
            uint64_t v[kMaxP];
#pragma unroll
            for (int w = 0; w < kMaxP; ++w) v[w] = w < a.p ? vp[w] : 0;
            if (a.xpoly) shift_payload<kMaxP>(v, a.polys, a.d, 0ull - r);
#pragma unroll
            for (int w = 0; w < kMaxP; ++w) {
                if (w >= a.p) break;
                dealer_rand(tl, a.rk, ge, SLOT_LUT_C + w, lo, hi);
                const uint64_t c0 = lo & a.mask;
                put(a.lut_c + (size_t)w * a.s8, c0, (v[w] - c0) & a.mask);
            }
        }
        dealer_rand(tl, a.rk, ge, SLOT_RIN, lo, hi);
        put(a.rin, lo & a.mask, (r - (lo & a.mask)) & a.mask);
        if (a.mask_output)
            for (int j = 0; j < a.n_out_a; ++j) {
                dealer_rand(tl, a.rk, ge, SLOT_ROUT + j, lo, hi);
                const uint64_t ro = a.r_out[(size_t)j * a.count + e] & a.mask, s0 = lo & a.mask;
                put(a.rout + (size_t)j * a.s8, s0, (ro - s0) & a.mask);
            }
        for (int t = 0; t < a.n_ka; ++t) {                                 // kappa^A = rep(r) >> arg
            dealer_rand(tl, a.rk, ge, SLOT_KA + t, lo, hi);
            uint64_t val = 0;
            if (a.ka_kind[t] == FUSEFSS_KA_R_SHR) val = a.ka_arg[t] >= 64 ? 0ull : r >> a.ka_arg[t];
            const uint64_t s0 = lo & a.mask;
            put(a.ka + (size_t)t * a.s8, s0, ((val & a.mask) - s0) & a.mask);
        }
        {                                                                  // variant 1 + bit 2: shares of (-r)^t, t = 1..d
            uint64_t pw = 1;
            for (int t = 1; t <= a.n_rpow; ++t) {
                pw = (pw * (0ull - r)) & a.mask;
                dealer_rand(tl, a.rk, ge, 0x5400 + t, lo, hi);
                const uint64_t s0 = lo & a.mask;
                put(a.rpow + (size_t)(t - 1) * a.s8, s0, (pw - s0) & a.mask);
            }
        }
        const int n_kb = a.n_carry + a.n_kb_spec;
        if (n_kb > 0) {
            uint64_t kbits = 0;
            int ci = 0;
            for (int t = 0; t < a.T; ++t) {                                // w_t = I[r_k + beta >= 2^k]  (Lemma 4.3, G3)
                if (!a.atom[t].is_theta) continue;
                const int k = a.atom[t].k;
                const uint64_t km = k >= 64 ? ~0ull : ((1ull << k) - 1ull);
                const uint64_t rk_ = r & km, sum = rk_ + a.atom[t].beta;
                const uint64_t w = k >= 64 ? (uint64_t)(sum < rk_) : (sum >> k) & 1ull;
                kbits |= w << ci++;
            }
            for (int t = 0; t < a.n_kb_spec; ++t) {
                uint64_t bit = 0;
                if (a.kb_kind[t] == FUSEFSS_KB_R_BIT) bit = (r >> a.kb_arg[t]) & 1ull;
                kbits |= bit << (a.n_carry + t);
            }
            dealer_rand(tl, a.rk, ge, SLOT_KB, lo, hi);
            const uint64_t s0 = lo & (n_kb >= 64 ? ~0ull : ((1ull << n_kb) - 1ull));
            put(a.kb, s0, kbits ^ s0);
        }
        int bv_word = 0;
        for (int i = 0; i < a.MA; ++i) {                                   // Beaver triple (a, b, c = ab)
            dealer_rand(tl, a.rk, ge, SLOT_BV_AB + i, lo, hi);
            const uint64_t ta = lo & a.mask, tb = hi & a.mask, tc = (ta * tb) & a.mask;
            dealer_rand(tl, a.rk, ge, SLOT_BV_AB0 + i, lo, hi);
            const uint64_t a0 = lo & a.mask, b0 = hi & a.mask;
            dealer_rand(tl, a.rk, ge, SLOT_BV_C0 + i, lo, hi);
            const uint64_t c0 = lo & a.mask;
            const size_t o = a.beaver + (size_t)bv_word * a.s8;
            if ((a.ma_is_x >> i) & 1ull) {
                const uint64_t cx = (tb * r) & a.mask;
                put(o, b0, (tb - b0) & a.mask);
                put(o + a.s8, c0, (cx - c0) & a.mask);
                bv_word += 2;
                continue;
            }
            bv_word += 3;
            put(o, a0, (ta - a0) & a.mask);
            put(o + a.s8, b0, (tb - b0) & a.mask);
            put(o + 2 * a.s8, c0, (tc - c0) & a.mask);
        }
        if (a.MB > 0) {                                                    // AND triples, gate i = bit i
            const uint64_t bm = a.MB >= 64 ? ~0ull : ((1ull << a.MB) - 1ull);
            dealer_rand(tl, a.rk, ge, SLOT_AND_AB, lo, hi);
            const uint64_t ta = lo & bm, tb = hi & bm, tc = ta & tb;
            dealer_rand(tl, a.rk, ge, SLOT_AND_AB0, lo, hi);
            const uint64_t a0 = lo & bm, b0 = hi & bm;
            dealer_rand(tl, a.rk, ge, SLOT_AND_C0, lo, hi);
            const uint64_t c0 = lo & bm;
            put(a.andt, a0, ta ^ a0);
            put(a.andt + a.s8, b0, tb ^ b0);
            put(a.andt + 2 * a.s8, c0, tc ^ c0);
        }
        if (a.GMIX > 0) {                                                  // B2A pairs (<rho>, [rho])
            const uint64_t bm = a.GMIX >= 64 ? ~0ull : ((1ull << a.GMIX) - 1ull);
            dealer_rand(tl, a.rk, ge, SLOT_B2A, lo, hi);
            const uint64_t rho = lo & bm, rho0 = hi & bm;
            put(a.b2a_bits, rho0, rho ^ rho0);
            for (int i = 0; i < a.GMIX; ++i) {
                dealer_rand(tl, a.rk, ge, SLOT_B2A_A0 + i, lo, hi);
                const uint64_t s0 = lo & a.mask, val = (rho >> i) & 1ull;
                put(a.b2a_a + (size_t)i * a.s8, s0, (val - s0) & a.mask);
            }
        }
        if (a.GA2B > 0) {                                                  // A2B (DESIGN 15): [rho_i] and <bit_j(rho_i)>; the keys f_{rho_i mod 2^j, 1} are k_gen_bit's
            uint64_t rbits = 0;
            for (int i = 0; i < a.GA2B; ++i) {
                dealer_rand(tl, a.rk, ge, SLOT_A2B_RHO + i, lo, hi);
                const uint64_t rho = lo & a.mask;
                dealer_rand(tl, a.rk, ge, SLOT_A2B_RHO0 + i, lo, hi);
                const uint64_t s0 = lo & a.mask;
                put(a.a2b_rho + (size_t)i * a.s8, s0, (rho - s0) & a.mask);
                rbits |= ((rho >> a.a2b_bit[i]) & 1ull) << i;
            }
            dealer_rand(tl, a.rk, ge, SLOT_A2B_BITS, lo, hi);
            const uint64_t b0 = lo & ((1ull << a.GA2B) - 1ull);
            put(a.a2b_bits, b0, rbits ^ b0);
        }
    }
}

__global__ void __launch_bounds__(kGenThreads, 1) k_gen_misc(const __grid_constant__ GenMiscArgs a) {
    extern __shared__ uint32_t sT[];
    gen_misc_body(a, aes_fill_tables(sT));
}

// ---------------------------------------------------------------------------------------------------
// The whole dealer step of a TINY tensor in ONE launch: bit trees, lookup trees (quad-lane) and share splitting run one after
// the other on the same persistent CTAs, with one table fill (a launch costs 9-10 us of launch + fill, profiles/r2u_small_split.md,
// which is most of a 4,096-element dealer pass).  The three parts write disjoint key sections, so no barrier separates them.
// ---------------------------------------------------------------------------------------------------
struct GenTinyArgs { GenBitArgs bit; GenVecArgs vec; GenMiscArgs misc; int has_bit, has_vec; };

template <int P>
__global__ void __launch_bounds__(kGenThreads, 1) k_gen_tiny(const __grid_constant__ GenTinyArgs a) {
    extern __shared__ uint32_t sT[];
    const uint32_t tl = aes_fill_tables(sT);
    if (a.has_bit) gen_bit_body(a.bit, tl);
    if (a.has_vec) gen_vec_quad_body<P>(a.vec, tl);
    gen_misc_body(a.misc, tl);
}

}  // namespace fsk
