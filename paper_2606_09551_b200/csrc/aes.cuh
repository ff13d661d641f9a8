// aes.cuh -- fixed-key AES-128 PRG core for sm_100a.
//
// T-table AES with T0..T3 in shared memory, REPLICATED PER BANK so that the 32 lanes of a warp always hit 32
// different banks: every LDS.32 is one conflict-free wavefront whatever the (secret-dependent) indices are.
// 160 lookups per block.  Layout chosen so that ONE PRMT builds the address of a lookup: entry x of a table
// sits at shared-window offset  block*65536 + x*256 + half*128 + lane*4  (T0/T1 = halves of block 1, T2/T3 =
// halves of block 2), so address = PRMT(state word, tl) = [tl.b0 | state byte k << 8 | tl.b2 | tl.b3] with
// tl = 0x00010000 | lane*4, and (block, half) ride in the LDS immediate.  Per round and block: 16 PRMT + 16 LDS +
// 8 LOP3 (the first version of this core used SHF + LOP3 + IMAD per lookup and was issue-bound; no profile of it is kept).
// State: 4 little-endian 32-bit words = the 4 columns (FIPS-197 3.4: byte r of word c is s[r][c]).
#pragma once
#include <cstdint>
#include <cstring>

namespace fsk {

#ifndef FFS_AES_UNROLL
#define FFS_AES_UNROLL 1          // rounds unrolled per loop trip (1, 3 or 9); chosen by measurement
#endif

constexpr int kAesUnroll = FFS_AES_UNROLL;
constexpr int kNumPrgKeys = 5;    // K_0 (children) + K_1..K_4 (payload blocks, p <= 8)

__constant__ uint32_t c_T0[256];                 // T0[x] = 2S | S<<8 | S<<16 | 3S<<24
__constant__ uint32_t c_rk[kNumPrgKeys][44];     // expanded K_i = (i, 01, .., 0f)

struct RoundKeys { uint32_t w[44]; };            // an expanded run-time key (dealer randomness, DESIGN 4.5)

// ---------------------------------------------------------------------------------------------------
// host side: S-box from log/antilog tables over GF(2^8) with generator 3, key expansion (FIPS-197 5.2)
// ---------------------------------------------------------------------------------------------------
struct HostAes {
    uint8_t sbox[256];
    uint32_t T0[256];
    HostAes() {
        uint8_t exp3[256], log3[256];
        uint8_t v = 1;
        for (int i = 0; i < 255; ++i) {
            exp3[i] = v; log3[v] = (uint8_t)i;
            uint8_t dbl = (uint8_t)((v << 1) ^ ((v & 0x80) ? 0x1b : 0));
            v = (uint8_t)(dbl ^ v);                                   // v *= 3
        }
        exp3[255] = exp3[0]; log3[0] = 0;
        for (int x = 0; x < 256; ++x) {
            uint8_t inv = x ? exp3[(255 - log3[x]) % 255] : 0;
            uint8_t s = inv, acc = inv;
            for (int k = 0; k < 4; ++k) { s = (uint8_t)((s << 1) | (s >> 7)); acc ^= s; }
            sbox[x] = (uint8_t)(acc ^ 0x63);
        }
        for (int x = 0; x < 256; ++x) {
            uint32_t s = sbox[x], s2 = ((s << 1) ^ ((s & 0x80) ? 0x11b : 0)) & 0xff, s3 = s2 ^ s;
            T0[x] = s2 | (s << 8) | (s << 16) | (s3 << 24);
        }
    }
    void expand(const uint8_t key[16], uint32_t w[44]) const {
        for (int i = 0; i < 4; ++i) std::memcpy(&w[i], key + 4 * i, 4);          // little-endian words
        uint32_t rcon = 1;
        for (int i = 4; i < 44; ++i) {
            uint32_t t = w[i - 1];
            if ((i & 3) == 0) {
                t = (t >> 8) | (t << 24);                                          // RotWord on LE bytes
                t = (uint32_t)sbox[t & 0xff] | ((uint32_t)sbox[(t >> 8) & 0xff] << 8) |
                    ((uint32_t)sbox[(t >> 16) & 0xff] << 16) | ((uint32_t)sbox[t >> 24] << 24);
                t ^= rcon;
                rcon = ((rcon << 1) ^ ((rcon & 0x80) ? 0x11b : 0)) & 0xff;
            }
            w[i] = w[i - 4] ^ t;
        }
    }
};

// ---------------------------------------------------------------------------------------------------
// device side
// ---------------------------------------------------------------------------------------------------
// Dynamic shared memory request: the tables occupy window offsets [65536, 196608); the dynamic region starts at
// a small offset B0 (reserved/static shared memory), so asking for 192 KB always covers them.
constexpr size_t kAesSmemBytes = 3 * 65536;

// Fills the tables and returns tl (= 0x00010000 | lane*4), produced AFTER the barrier by a volatile asm so that
// no table lookup (all of which consume tl) can be scheduled above it.
__device__ __forceinline__ uint32_t aes_fill_tables(uint32_t *dyn_smem) {
    const uint32_t b0 = (uint32_t)__cvta_generic_to_shared(dyn_smem);
    char *win0 = reinterpret_cast<char *>(dyn_smem) - b0;                  // generic address of window offset 0
    for (int i = threadIdx.x; i < 256 * 32; i += blockDim.x) {            // one constant load feeds the four rotations
        const int x = i >> 5, ln = i & 31;
        const uint32_t v = c_T0[x];
        char *p = win0 + 65536u + (uint32_t)x * 256u + (uint32_t)ln * 4u;
        *reinterpret_cast<uint32_t *>(p) = v;                                         // T0
        *reinterpret_cast<uint32_t *>(p + 128) = __funnelshift_l(v, v, 8);            // T1 = T0 rotated left by 8 bits
        *reinterpret_cast<uint32_t *>(p + 65536) = __funnelshift_l(v, v, 16);         // T2
        *reinterpret_cast<uint32_t *>(p + 65536 + 128) = __funnelshift_l(v, v, 24);   // T3
    }
    __syncthreads();
    uint32_t tl;
    asm volatile("mov.u32 %0, %1;" : "=r"(tl) : "r"(0x00010000u | ((threadIdx.x & 31u) << 2)) : "memory");
    return tl;
}

// T_TAB[ byte K of w ]
template <int TAB, int K>
__device__ __forceinline__ uint32_t tlu(uint32_t tl, uint32_t w) {
    uint32_t v;
    asm("{\n\t.reg .b32 a;\n\tprmt.b32 a, %1, %2, %3;\n\tld.shared.u32 %0, [a+%4];\n\t}"
        : "=r"(v) : "r"(w), "r"(tl), "n"(0x7604 | (K << 4)), "n"((TAB >> 1) * 65536 + (TAB & 1) * 128));
    return v;
}

__device__ __forceinline__ void aes_round(uint32_t (&s)[4], uint32_t tl, uint32_t k0, uint32_t k1, uint32_t k2, uint32_t k3) {
    uint32_t t0 = tlu<0, 0>(tl, s[0]) ^ tlu<1, 1>(tl, s[1]) ^ tlu<2, 2>(tl, s[2]) ^ tlu<3, 3>(tl, s[3]) ^ k0;
    uint32_t t1 = tlu<0, 0>(tl, s[1]) ^ tlu<1, 1>(tl, s[2]) ^ tlu<2, 2>(tl, s[3]) ^ tlu<3, 3>(tl, s[0]) ^ k1;
    uint32_t t2 = tlu<0, 0>(tl, s[2]) ^ tlu<1, 1>(tl, s[3]) ^ tlu<2, 2>(tl, s[0]) ^ tlu<3, 3>(tl, s[1]) ^ k2;
    uint32_t t3 = tlu<0, 0>(tl, s[3]) ^ tlu<1, 1>(tl, s[0]) ^ tlu<2, 2>(tl, s[1]) ^ tlu<3, 3>(tl, s[2]) ^ k3;
    s[0] = t0; s[1] = t1; s[2] = t2; s[3] = t3;
}

// final round: SubBytes + ShiftRows (+ AddRoundKey by the caller).  S[x] = byte 0 of T2 = byte 1 of T3 = byte 2
// of T0 = byte 3 of T1, so the column is assembled with three PRMTs.
__device__ __forceinline__ uint32_t aes_last_col(uint32_t tl, uint32_t a, uint32_t b, uint32_t c, uint32_t d) {
    const uint32_t va = tlu<2, 0>(tl, a), vb = tlu<3, 1>(tl, b), vc = tlu<0, 2>(tl, c), vd = tlu<1, 3>(tl, d);
    const uint32_t lo = __byte_perm(va, vb, 0x3250);      // [va.b0, vb.b1, -, -]
    const uint32_t hi = __byte_perm(vc, vd, 0x7210);      // [-, -, vc.b2, vd.b3]
    return __byte_perm(lo, hi, 0x7610);
}
__device__ __forceinline__ void aes_last(uint32_t (&s)[4], uint32_t tl, uint32_t k0, uint32_t k1, uint32_t k2, uint32_t k3) {
    uint32_t t0 = aes_last_col(tl, s[0], s[1], s[2], s[3]) ^ k0;
    uint32_t t1 = aes_last_col(tl, s[1], s[2], s[3], s[0]) ^ k1;
    uint32_t t2 = aes_last_col(tl, s[2], s[3], s[0], s[1]) ^ k2;
    uint32_t t3 = aes_last_col(tl, s[3], s[0], s[1], s[2]) ^ k3;
    s[0] = t0; s[1] = t1; s[2] = t2; s[3] = t3;
}

// NI inputs x NK keys (K_KFIRST .. K_{KFIRST+NK-1}) in lock-step: out[i][k] = AES_{K}(x_i) ^ x_i  (the PRG of 4.1).
// SHARE = 1 asserts that the NI inputs differ only in byte 0 of word 0 (the tweak of ONE seed).  The PRG keys
// K_i = (i, 01, .., 0f) differ only in byte 0 too, so after the initial AddRoundKey all NI*NK states agree except
// in that byte, which feeds a single lookup of round 1 (column 0, T0): the other 15 lookups of round 1 are done
// once and shared -- 15 + NI*NK lookups instead of 16*NI*NK.  SHARE = 2: the inputs are unrelated seeds (several points
// walked in lock-step), the NK keys of EACH input share their 15 lookups.  SHARE = 0: nothing is shared.
// UNR = rounds unrolled per loop trip: 1 for the register-hungry kernels (k_gen_vec, k_eval_p3), 3 where it measured
// faster (k_eval_sp, k_gen_bit): profiles/r1l_unroll.md.
template <int NI, int NK, int KFIRST, int SHARE = 0, int UNR = kAesUnroll>
__device__ __forceinline__ void prg_blocks(uint32_t tl, const uint32_t (&x)[NI][4], uint32_t (&out)[NI][NK][4]) {
    if (SHARE == 1 && NI * NK > 1) {
        uint32_t w[4];
#pragma unroll
        for (int c = 0; c < 4; ++c) w[c] = x[0][c] ^ c_rk[KFIRST][c];
        const uint32_t c0 = tlu<1, 1>(tl, w[1]) ^ tlu<2, 2>(tl, w[2]) ^ tlu<3, 3>(tl, w[3]);
        const uint32_t c1 = tlu<0, 0>(tl, w[1]) ^ tlu<1, 1>(tl, w[2]) ^ tlu<2, 2>(tl, w[3]) ^ tlu<3, 3>(tl, w[0]);
        const uint32_t c2 = tlu<0, 0>(tl, w[2]) ^ tlu<1, 1>(tl, w[3]) ^ tlu<2, 2>(tl, w[0]) ^ tlu<3, 3>(tl, w[1]);
        const uint32_t c3 = tlu<0, 0>(tl, w[3]) ^ tlu<1, 1>(tl, w[0]) ^ tlu<2, 2>(tl, w[1]) ^ tlu<3, 3>(tl, w[2]);
#pragma unroll
        for (int i = 0; i < NI; ++i)
#pragma unroll
            for (int k = 0; k < NK; ++k) {
                out[i][k][0] = c0 ^ tlu<0, 0>(tl, x[i][0] ^ c_rk[KFIRST + k][0]) ^ c_rk[KFIRST + k][4];
                out[i][k][1] = c1 ^ c_rk[KFIRST + k][5];
                out[i][k][2] = c2 ^ c_rk[KFIRST + k][6];
                out[i][k][3] = c3 ^ c_rk[KFIRST + k][7];
            }
    } else if (SHARE == 2 && NK > 1) {
#pragma unroll
        for (int i = 0; i < NI; ++i) {
            uint32_t w[4];
#pragma unroll
            for (int c = 0; c < 4; ++c) w[c] = x[i][c] ^ c_rk[KFIRST][c];
            const uint32_t c0 = tlu<1, 1>(tl, w[1]) ^ tlu<2, 2>(tl, w[2]) ^ tlu<3, 3>(tl, w[3]);
            const uint32_t c1 = tlu<0, 0>(tl, w[1]) ^ tlu<1, 1>(tl, w[2]) ^ tlu<2, 2>(tl, w[3]) ^ tlu<3, 3>(tl, w[0]);
            const uint32_t c2 = tlu<0, 0>(tl, w[2]) ^ tlu<1, 1>(tl, w[3]) ^ tlu<2, 2>(tl, w[0]) ^ tlu<3, 3>(tl, w[1]);
            const uint32_t c3 = tlu<0, 0>(tl, w[3]) ^ tlu<1, 1>(tl, w[0]) ^ tlu<2, 2>(tl, w[1]) ^ tlu<3, 3>(tl, w[2]);
#pragma unroll
            for (int k = 0; k < NK; ++k) {
                out[i][k][0] = c0 ^ tlu<0, 0>(tl, x[i][0] ^ c_rk[KFIRST + k][0]) ^ c_rk[KFIRST + k][4];
                out[i][k][1] = c1 ^ c_rk[KFIRST + k][5];
                out[i][k][2] = c2 ^ c_rk[KFIRST + k][6];
                out[i][k][3] = c3 ^ c_rk[KFIRST + k][7];
            }
        }
    } else {
#pragma unroll
        for (int i = 0; i < NI; ++i)
#pragma unroll
            for (int k = 0; k < NK; ++k) {
#pragma unroll
                for (int c = 0; c < 4; ++c) out[i][k][c] = x[i][c] ^ c_rk[KFIRST + k][c];
                aes_round(out[i][k], tl, c_rk[KFIRST + k][4], c_rk[KFIRST + k][5], c_rk[KFIRST + k][6], c_rk[KFIRST + k][7]);
            }
    }
#pragma unroll UNR
    for (int r = 2; r < 10; ++r) {
#pragma unroll
        for (int i = 0; i < NI; ++i)
#pragma unroll
            for (int k = 0; k < NK; ++k)
                aes_round(out[i][k], tl, c_rk[KFIRST + k][4 * r], c_rk[KFIRST + k][4 * r + 1],
                          c_rk[KFIRST + k][4 * r + 2], c_rk[KFIRST + k][4 * r + 3]);
    }
#pragma unroll
    for (int i = 0; i < NI; ++i)
#pragma unroll
        for (int k = 0; k < NK; ++k) {
            aes_last(out[i][k], tl, c_rk[KFIRST + k][40], c_rk[KFIRST + k][41], c_rk[KFIRST + k][42], c_rk[KFIRST + k][43]);
#pragma unroll
            for (int c = 0; c < 4; ++c) out[i][k][c] ^= x[i][c];
        }
}

// plain AES-128 with a run-time expanded key (no feed-forward): R(e, slot) of DESIGN 4.5
__device__ __forceinline__ void aes_encrypt_rk(uint32_t tl, const RoundKeys &rk, uint32_t (&s)[4]) {
#pragma unroll
    for (int c = 0; c < 4; ++c) s[c] ^= rk.w[c];
#pragma unroll 1
    for (int r = 1; r < 10; ++r) aes_round(s, tl, rk.w[4 * r], rk.w[4 * r + 1], rk.w[4 * r + 2], rk.w[4 * r + 3]);
    aes_last(s, tl, rk.w[40], rk.w[41], rk.w[42], rk.w[43]);
}

}  // namespace fsk
