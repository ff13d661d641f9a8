// bitslice.cuh -- a bitsliced AES-128 core, built ONLY to time it against the T-table core (DESIGN 5.2; north_star: "shared-memory
// T-tables or a bitsliced design chosen by measurement").  It is not on the hot path.
// One thread holds 32 blocks as 128 bit-planes: p[b][i] = bit i of state byte b (b = r + 4c, FIPS-197 3.4) for its 32 blocks, so
// every instruction is a 32-bit logic op on registers -- no table, no shared memory.  SubBytes = the generated composite-field
// circuit (bitslice_sbox.cuh, 152 XOR + 36 AND per byte; the smallest published circuit has 113 gates), ShiftRows = register
// moves, MixColumns = xtime on planes, AddRoundKey = XOR with all-ones / all-zero words from constant memory.
#pragma once
#include "bitslice_sbox.cuh"

namespace fsk {

__constant__ uint32_t c_bs_rk[11][128];      // round key bit (8 b + i) of round r, replicated to a 32-bit mask

__device__ __forceinline__ void bs_add_round_key(uint32_t (&p)[16][8], int r) {
#pragma unroll
    for (int b = 0; b < 16; ++b)
#pragma unroll
        for (int i = 0; i < 8; ++i) p[b][i] ^= c_bs_rk[r][8 * b + i];
}

__device__ __forceinline__ void bs_shift_rows(uint32_t (&p)[16][8]) {
#pragma unroll
    for (int i = 0; i < 8; ++i) {                 // row r (bytes r, r+4, r+8, r+12) rotates left by r columns
        uint32_t t = p[1][i]; p[1][i] = p[5][i]; p[5][i] = p[9][i]; p[9][i] = p[13][i]; p[13][i] = t;
        t = p[2][i]; p[2][i] = p[10][i]; p[10][i] = t; t = p[6][i]; p[6][i] = p[14][i]; p[14][i] = t;
        t = p[15][i]; p[15][i] = p[11][i]; p[11][i] = p[7][i]; p[7][i] = p[3][i]; p[3][i] = t;
    }
}

// out_r = xtime(a_r ^ a_{r+1}) ^ a_{r+1} ^ a_{r+2} ^ a_{r+3}  (= 2 a_r + 3 a_{r+1} + a_{r+2} + a_{r+3}), per column, in place
__device__ __forceinline__ void bs_mix_columns(uint32_t (&p)[16][8]) {
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        uint32_t a[4][8], all[8];
#pragma unroll
        for (int r = 0; r < 4; ++r)
#pragma unroll
            for (int i = 0; i < 8; ++i) a[r][i] = p[r + 4 * c][i];
#pragma unroll
        for (int i = 0; i < 8; ++i) all[i] = a[0][i] ^ a[1][i] ^ a[2][i] ^ a[3][i];
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            uint32_t t[8];
#pragma unroll
            for (int i = 0; i < 8; ++i) t[i] = a[r][i] ^ a[(r + 1) & 3][i];
            // xtime(t): shift left by one bit position, reduce by x^8 = x^4 + x^3 + x + 1
            uint32_t x2[8] = {t[7], t[0] ^ t[7], t[1], t[2] ^ t[7], t[3] ^ t[7], t[4], t[5], t[6]};
#pragma unroll
            for (int i = 0; i < 8; ++i) p[r + 4 * c][i] = x2[i] ^ all[i] ^ a[r][i];
        }
    }
}

__device__ __forceinline__ void bs_encrypt(uint32_t (&p)[16][8]) {
    bs_add_round_key(p, 0);
#pragma unroll 1
    for (int r = 1; r <= 10; ++r) {
#pragma unroll
        for (int b = 0; b < 16; ++b) bitslice_sbox(p[b]);
        bs_shift_rows(p);
        if (r < 10) bs_mix_columns(p);
        bs_add_round_key(p, r);
    }
}

struct BsProbeArgs { uint4 *out; size_t threads; int iters; };
// throughput probe: every thread chains `iters` encryptions of its 32 blocks (ciphertext -> next plaintext)
__global__ void __launch_bounds__(256, 1) k_bitslice_probe(const BsProbeArgs a) {
    for (size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x; t < a.threads; t += (size_t)gridDim.x * blockDim.x) {
        uint32_t p[16][8];
#pragma unroll
        for (int b = 0; b < 16; ++b)
#pragma unroll
            for (int i = 0; i < 8; ++i) p[b][i] = (uint32_t)t * 2654435761u + (uint32_t)(8 * b + i) * 40503u;
        for (int it = 0; it < a.iters; ++it) bs_encrypt(p);
        uint32_t acc[4] = {0, 0, 0, 0};
#pragma unroll
        for (int b = 0; b < 16; ++b)
#pragma unroll
            for (int i = 0; i < 8; ++i) acc[(b + i) & 3] ^= p[b][i];
        a.out[t] = make_uint4(acc[0], acc[1], acc[2], acc[3]);
    }
}

struct BsKatArgs { const uint8_t *in; uint8_t *out; };    // device: 32 blocks of 16 bytes each
// known-answer path: one thread packs 32 blocks into planes, encrypts them once, unpacks
__global__ void k_bitslice_kat(const BsKatArgs a) {
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    uint32_t p[16][8];
#pragma unroll
    for (int b = 0; b < 16; ++b)
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            uint32_t w = 0;
            for (int k = 0; k < 32; ++k) w |= (uint32_t)((a.in[16 * k + b] >> i) & 1u) << k;
            p[b][i] = w;
        }
    bs_encrypt(p);
    for (int k = 0; k < 32; ++k)
#pragma unroll
        for (int b = 0; b < 16; ++b) {
            uint32_t v = 0;
#pragma unroll
            for (int i = 0; i < 8; ++i) v |= ((p[b][i] >> k) & 1u) << i;
            a.out[16 * k + b] = (uint8_t)v;
        }
}

}  // namespace fsk
