// aes.cuh -- fixed-key AES-128 PRG core for sm_100a.
//
// T-table AES with the tables in shared memory, REPLICATED PER BANK: entry x of table k lives at word
// (k*256 + x)*32 + lane, so the 32 lanes of a warp always hit 32 different banks and every LDS.32 is one
// conflict-free wavefront whatever the (secret-dependent, random) indices are.  160 lookups per block.
// NTAB = 4 keeps T0..T3 (128 KB); NTAB = 1 keeps T0 only (32 KB) and rotates with PRMT.
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
template <int NTAB>
__device__ __forceinline__ void aes_fill_tables(uint32_t *sT) {
    for (int i = threadIdx.x; i < NTAB * 256 * 32; i += blockDim.x) {
        uint32_t v = c_T0[(i >> 5) & 255];
        int rot = (i >> 13) * 8;                                      // table k = T0 rotated left by 8k bits
        sT[i] = __funnelshift_l(v, v, rot);
    }
    __syncthreads();
}

template <int NTAB> constexpr size_t aes_smem_bytes() { return (size_t)NTAB * 256 * 32 * 4; }

template <int K> __device__ __forceinline__ uint32_t byte_of(uint32_t w) {
    return K == 0 ? (w & 0xffu) : K == 3 ? (w >> 24) : ((w >> (8 * K)) & 0xffu);
}

// lookup of table TAB at the byte K of w; `tl` = shared table base already offset by the lane
template <int NTAB, int TAB, int K>
__device__ __forceinline__ uint32_t tlu(const uint32_t *tl, uint32_t w) {
    if (NTAB == 4) return tl[TAB * 8192 + byte_of<K>(w) * 32];
    uint32_t v = tl[byte_of<K>(w) * 32];
    return TAB == 0 ? v : TAB == 1 ? __byte_perm(v, v, 0x2103) : TAB == 2 ? __byte_perm(v, v, 0x1032)
                                                                          : __byte_perm(v, v, 0x0321);
}

template <int NTAB>
__device__ __forceinline__ void aes_round(uint32_t (&s)[4], const uint32_t *tl, uint32_t k0, uint32_t k1,
                                          uint32_t k2, uint32_t k3) {
    uint32_t t0 = tlu<NTAB, 0, 0>(tl, s[0]) ^ tlu<NTAB, 1, 1>(tl, s[1]) ^ tlu<NTAB, 2, 2>(tl, s[2]) ^ tlu<NTAB, 3, 3>(tl, s[3]) ^ k0;
    uint32_t t1 = tlu<NTAB, 0, 0>(tl, s[1]) ^ tlu<NTAB, 1, 1>(tl, s[2]) ^ tlu<NTAB, 2, 2>(tl, s[3]) ^ tlu<NTAB, 3, 3>(tl, s[0]) ^ k1;
    uint32_t t2 = tlu<NTAB, 0, 0>(tl, s[2]) ^ tlu<NTAB, 1, 1>(tl, s[3]) ^ tlu<NTAB, 2, 2>(tl, s[0]) ^ tlu<NTAB, 3, 3>(tl, s[1]) ^ k2;
    uint32_t t3 = tlu<NTAB, 0, 0>(tl, s[3]) ^ tlu<NTAB, 1, 1>(tl, s[0]) ^ tlu<NTAB, 2, 2>(tl, s[1]) ^ tlu<NTAB, 3, 3>(tl, s[2]) ^ k3;
    s[0] = t0; s[1] = t1; s[2] = t2; s[3] = t3;
}

// final round: SubBytes + ShiftRows + AddRoundKey; S[x] is byte 1 (and 2) of T0[x]
template <int NTAB>
__device__ __forceinline__ uint32_t aes_last_col(const uint32_t *tl, uint32_t a, uint32_t b, uint32_t c, uint32_t d) {
    if (NTAB == 4) {
        return (tl[2 * 8192 + byte_of<0>(a) * 32] & 0x000000ffu) | (tl[3 * 8192 + byte_of<1>(b) * 32] & 0x0000ff00u) |
               (tl[0 * 8192 + byte_of<2>(c) * 32] & 0x00ff0000u) | (tl[1 * 8192 + byte_of<3>(d) * 32] & 0xff000000u);
    }
    uint32_t va = tl[byte_of<0>(a) * 32], vb = tl[byte_of<1>(b) * 32], vc = tl[byte_of<2>(c) * 32], vd = tl[byte_of<3>(d) * 32];
    uint32_t lo = __byte_perm(va, vb, 0x0051);      // bytes: va.b1, vb.b1
    uint32_t hi = __byte_perm(vc, vd, 0x0051);
    return __byte_perm(lo, hi, 0x5410);
}
template <int NTAB>
__device__ __forceinline__ void aes_last(uint32_t (&s)[4], const uint32_t *tl, uint32_t k0, uint32_t k1, uint32_t k2, uint32_t k3) {
    uint32_t t0 = aes_last_col<NTAB>(tl, s[0], s[1], s[2], s[3]) ^ k0;
    uint32_t t1 = aes_last_col<NTAB>(tl, s[1], s[2], s[3], s[0]) ^ k1;
    uint32_t t2 = aes_last_col<NTAB>(tl, s[2], s[3], s[0], s[1]) ^ k2;
    uint32_t t3 = aes_last_col<NTAB>(tl, s[3], s[0], s[1], s[2]) ^ k3;
    s[0] = t0; s[1] = t1; s[2] = t2; s[3] = t3;
}

// NI inputs x NK keys (K_KFIRST .. K_{KFIRST+NK-1}) in lock-step: out[i][k] = AES_{K}(x_i) ^ x_i  (the PRG of 4.1)
template <int NTAB, int NI, int NK, int KFIRST>
__device__ __forceinline__ void prg_blocks(const uint32_t *tl, const uint32_t (&x)[NI][4], uint32_t (&out)[NI][NK][4]) {
#pragma unroll
    for (int i = 0; i < NI; ++i)
#pragma unroll
        for (int k = 0; k < NK; ++k)
#pragma unroll
            for (int c = 0; c < 4; ++c) out[i][k][c] = x[i][c] ^ c_rk[KFIRST + k][c];
#pragma unroll kAesUnroll
    for (int r = 1; r < 10; ++r) {
#pragma unroll
        for (int i = 0; i < NI; ++i)
#pragma unroll
            for (int k = 0; k < NK; ++k)
                aes_round<NTAB>(out[i][k], tl, c_rk[KFIRST + k][4 * r], c_rk[KFIRST + k][4 * r + 1],
                                c_rk[KFIRST + k][4 * r + 2], c_rk[KFIRST + k][4 * r + 3]);
    }
#pragma unroll
    for (int i = 0; i < NI; ++i)
#pragma unroll
        for (int k = 0; k < NK; ++k) {
            aes_last<NTAB>(out[i][k], tl, c_rk[KFIRST + k][40], c_rk[KFIRST + k][41], c_rk[KFIRST + k][42], c_rk[KFIRST + k][43]);
#pragma unroll
            for (int c = 0; c < 4; ++c) out[i][k][c] ^= x[i][c];
        }
}

// plain AES-128 with a run-time expanded key (no feed-forward): R(e, slot) of DESIGN 4.5
template <int NTAB>
__device__ __forceinline__ void aes_encrypt_rk(const uint32_t *tl, const RoundKeys &rk, uint32_t (&s)[4]) {
#pragma unroll
    for (int c = 0; c < 4; ++c) s[c] ^= rk.w[c];
#pragma unroll 1
    for (int r = 1; r < 10; ++r) aes_round<NTAB>(s, tl, rk.w[4 * r], rk.w[4 * r + 1], rk.w[4 * r + 2], rk.w[4 * r + 3]);
    aes_last<NTAB>(s, tl, rk.w[40], rk.w[41], rk.w[42], rk.w[43]);
}

}  // namespace fsk
