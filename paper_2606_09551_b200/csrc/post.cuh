// post.cuh -- share-based post-processing (a7): online steps 4-6.
// Protocol 2, predicate bits = atoms xor carries (Lemma 4.3), Boolean AND with bit triples, B2A,
// Horner with Beaver multiplications, optional masked output yhat = y + r_out.
// Subprotocol formulas and message layout: DESIGN 4.6.  One lane per element interprets the compiled
// straight-line program (program.h Ins) out of global memory (uniform across the warp); arithmetic registers
// live in a small per-thread array, bit registers in one 64-bit word.
// A2B nodes (DESIGN 15): bit 0 of a shared value is local; bit j >= 1 opens ehat = e + rho and evaluates the dealer's
// j-bit comparison key at ehat mod 2^j: bit_j(e) = bit_j(ehat) ^ bit_j(rho) ^ I[ehat mod 2^j < rho mod 2^j].  Programs with such
// nodes run the <true> instantiations: persistent CTAs with the PRG tables in shared memory (grid-stride over elements).
#pragma once
#include "eval.cuh"
#include "program.h"

namespace fsk {

struct PostKeyOff {                                                                  // (rpow is read by the eval kernel only)
    size_t s8, rin, rout, ka, kb, beaver, andt, b2a_bits, b2a_a;
    size_t s16, a2b_rho, a2b_bits, a2b_root[kMaxA2B], a2b_cw[kMaxA2B], a2b_vb[kMaxA2B];
    int et, pad;
};

struct PostArgs {
    const Ins *ins; int n_ins;
    int party, round, rounds, mask_output, n_out_a, n_out_b, pad;
    const uint8_t *key; const uint64_t *xhat, *bits, *coeff;
    const uint8_t *msg_in; uint8_t *msg_out;
    uint64_t *y_out, *z_out;
    size_t count; uint64_t mask;
    PostKeyOff k;
    size_t round_off[kMaxRounds + 1];
    int round_arr[kMaxRounds];     // ring-element arrays opened in the round (the bit word follows them)
    int round_bits[kMaxRounds];
};

__device__ __forceinline__ uint64_t kld(const uint8_t *key, size_t off, size_t e) {
    return reinterpret_cast<const uint64_t *>(key + off)[e];
}

// one party, one round; stateless replay of earlier rounds from the two message buffers
template <bool A2B>
__global__ void __launch_bounds__(256) k_post_round(const __grid_constant__ PostArgs a) {
    extern __shared__ uint32_t sT[];
    uint32_t tl = 0;
    if (A2B) tl = aes_fill_tables(sT);
    for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < a.count; e += (size_t)gridDim.x * blockDim.x) {
    const uint64_t mask = a.mask, xh = a.xhat[e] & mask;
    const bool p0 = a.party == 0;
    uint64_t A[kMaxAReg];
    uint64_t Bw0 = 0, Bw1 = 0, zword = 0, outbits = 0;                       // 128 bit registers (kMaxBReg) in two words
    auto getb = [&](int r) -> uint64_t { return ((r < 64 ? Bw0 : Bw1) >> (r & 63)) & 1ull; };
    auto setb = [&](int r, uint64_t v) {
        const uint64_t m = 1ull << (r & 63), b = (v & 1ull) << (r & 63);
        if (r < 64) Bw0 = (Bw0 & ~m) | b; else Bw1 = (Bw1 & ~m) | b;
    };
    for (int pc = 0; pc < a.n_ins; ++pc) {
        const Ins o = a.ins[pc];
        switch (o.op) {
        case I_B_CONST: setb(o.dst, p0 ? o.imm : 0); break;
        case I_B_ATOM: setb(o.dst, a.bits[e] >> o.a); break;
        case I_B_KAPPA: setb(o.dst, kld(a.key, a.k.kb, e) >> o.a); break;
        case I_B_XHAT: setb(o.dst, p0 ? xh >> o.a : 0); break;
        case I_B_NOT: setb(o.dst, getb(o.a) ^ (p0 ? 1ull : 0ull)); break;
        case I_B_XOR: setb(o.dst, getb(o.a) ^ getb(o.b)); break;
        case I_B_ANDPUB: setb(o.dst, getb(o.a) & ((xh >> o.b) ^ o.imm)); break;
        case I_B_OUT: zword |= getb(o.a) << o.dst; break;
        case I_B_AND: {
            const uint64_t ta = (kld(a.key, a.k.andt, e) >> o.gate) & 1, tb = (kld(a.key, a.k.andt + a.k.s8, e) >> o.gate) & 1,
                           tc = (kld(a.key, a.k.andt + 2 * a.k.s8, e) >> o.gate) & 1;
            const uint64_t dm = getb(o.a) ^ ta, em = getb(o.b) ^ tb;
            const int q = o.round;
            if (q == a.round) outbits |= (dm << o.pos) | (em << (o.pos + 1));
            uint64_t res = 0;
            if (q < a.round) {
                const uint64_t other = kld(a.msg_in, a.round_off[q] + (size_t)a.round_arr[q] * a.k.s8, e);
                const uint64_t dd = dm ^ ((other >> o.pos) & 1), ee = em ^ ((other >> (o.pos + 1)) & 1);
                res = (p0 ? (dd & ee) : 0) ^ (dd & tb) ^ (ee & ta) ^ tc;
            }
            setb(o.dst, res);
            break; }
        case I_A_CONST: A[o.dst] = p0 ? (o.imm & mask) : 0; break;
        case I_A_X: { const uint64_t r = kld(a.key, a.k.rin, e); A[o.dst] = (p0 ? xh - r : 0ull - r) & mask; break; }
        case I_A_COEFF: A[o.dst] = a.coeff[(size_t)o.a * a.count + e] & mask; break;
        case I_A_KAPPA: A[o.dst] = kld(a.key, a.k.ka + (size_t)o.a * a.k.s8, e); break;
        case I_A_XHAT_SHR: A[o.dst] = p0 ? (o.a >= 64 ? 0ull : xh >> o.a) : 0ull; break;
        case I_A_ADD: A[o.dst] = (A[o.a] + A[o.b]) & mask; break;
        case I_A_SUB: A[o.dst] = (A[o.a] - A[o.b]) & mask; break;
        case I_A_MULC: A[o.dst] = (A[o.a] * o.imm) & mask; break;
        case I_A_MULXH: A[o.dst] = (A[o.a] * xh) & mask; break;          // share times the public xhat (DESIGN 11)
        case I_A_OUT:
            if (a.round == a.rounds) {
                uint64_t v = A[o.a];
                if (a.mask_output) v = (v + kld(a.key, a.k.rout + (size_t)o.dst * a.k.s8, e)) & mask;
                a.y_out[(size_t)o.dst * a.count + e] = v;
            }
            break;
        case I_A_MUL: {
            const size_t to = a.k.beaver + (size_t)o.imm * a.k.s8;
            const uint64_t ta = kld(a.key, to, e), tb = kld(a.key, to + a.k.s8, e), tc = kld(a.key, to + 2 * a.k.s8, e);
            const uint64_t em = (A[o.a] - ta) & mask, fm = (A[o.b] - tb) & mask;
            const int q = o.round;
            const size_t mo = a.round_off[q] + (size_t)o.pos * a.k.s8;
            if (q == a.round) {
                reinterpret_cast<uint64_t *>(a.msg_out + mo)[e] = em;
                reinterpret_cast<uint64_t *>(a.msg_out + mo + a.k.s8)[e] = fm;
            }
            uint64_t res = 0;
            if (q < a.round) {
                const uint64_t E = (em + kld(a.msg_in, mo, e)) & mask, F = (fm + kld(a.msg_in, mo + a.k.s8, e)) & mask;
                res = ((p0 ? E * F : 0) + E * tb + F * ta + tc) & mask;
            }
            A[o.dst] = res;
            break; }
        case I_A_MULX: {     // y * x, x = xhat - r_in: material (b, c = b r_in), open f = y - b; [yx]_b = xhat [y]_b - f [r_in]_b - [c]_b
            const size_t to = a.k.beaver + (size_t)o.imm * a.k.s8;
            const uint64_t tb = kld(a.key, to, e), tc = kld(a.key, to + a.k.s8, e);
            const uint64_t fm = (A[o.a] - tb) & mask;
            const int q = o.round;
            const size_t mo = a.round_off[q] + (size_t)o.pos * a.k.s8;
            if (q == a.round) reinterpret_cast<uint64_t *>(a.msg_out + mo)[e] = fm;
            uint64_t res = 0;
            if (q < a.round) {
                const uint64_t F = (fm + kld(a.msg_in, mo, e)) & mask;
                res = (xh * A[o.a] - F * kld(a.key, a.k.rin, e) - tc) & mask;
            }
            A[o.dst] = res;
            break; }
        case I_A_B2A: {
            const uint64_t rb = (kld(a.key, a.k.b2a_bits, e) >> o.gate) & 1, ra = kld(a.key, a.k.b2a_a + (size_t)o.gate * a.k.s8, e);
            const uint64_t mm = getb(o.a) ^ rb;
            const int q = o.round;
            if (q == a.round) outbits |= mm << o.pos;
            uint64_t res = 0;
            if (q < a.round) {
                const uint64_t other = kld(a.msg_in, a.round_off[q] + (size_t)a.round_arr[q] * a.k.s8, e);
                const uint64_t mu = mm ^ ((other >> o.pos) & 1);
                res = ((p0 ? mu : 0) + ra - 2 * mu * ra) & mask;
            }
            A[o.dst] = res;
            break; }
        case I_B_LSB: setb(o.dst, A[o.a]); break;                          // (e_0 + e_1) mod 2 = e_0 ^ e_1 on the low bit
        case I_B_A2B: {
            uint64_t res = 0;
            if (A2B) {
                const int q = o.round, j = (int)o.imm, g = o.gate;
                const uint64_t em = (A[o.a] + kld(a.key, a.k.a2b_rho + (size_t)g * a.k.s8, e)) & mask;
                const size_t mo = a.round_off[q] + (size_t)o.pos * a.k.s8;
                if (q == a.round) reinterpret_cast<uint64_t *>(a.msg_out + mo)[e] = em;
                if (q < a.round) {
                    const uint64_t E = (em + kld(a.msg_in, mo, e)) & mask;
                    const uint32_t c = bit_tree_eval<false>(tl, a.key, a.k.a2b_root[g], a.k.a2b_cw[g], a.k.a2b_vb[g], e, a.k.s16, j,
                                                            E << (64 - j), a.party, a.k.et);
                    res = (p0 ? (E >> j) : 0ull) ^ (kld(a.key, a.k.a2b_bits, e) >> g) ^ (uint64_t)c;
                }
            }
            setb(o.dst, res);
            break; }
        default: break;
        }
    }
    if (a.round < a.rounds && a.round_bits[a.round])
        reinterpret_cast<uint64_t *>(a.msg_out + a.round_off[a.round] + (size_t)a.round_arr[a.round] * a.k.s8)[e] = outbits;
    if (a.round == a.rounds && a.n_out_b > 0) a.z_out[e] = zword;
    }
}

struct PostFusedArgs {
    const Ins *ins; int n_ins;
    int mask_output, n_out_a, n_out_b;
    const uint8_t *key[2]; const uint64_t *xhat, *bits[2], *coeff[2];
    uint64_t *y_out[2], *z_out[2];
    size_t count; uint64_t mask;
    PostKeyOff k;
};

// both parties, all rounds, one pass: the openings are combined in registers instead of message buffers
template <bool A2B>
__global__ void __launch_bounds__(256) k_post_fused(const __grid_constant__ PostFusedArgs a) {
    extern __shared__ uint32_t sT[];
    uint32_t tl = 0;
    if (A2B) tl = aes_fill_tables(sT);
    for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < a.count; e += (size_t)gridDim.x * blockDim.x) {
    const uint64_t mask = a.mask, xh = a.xhat[e] & mask;
    uint64_t A[2][kMaxAReg];
    uint64_t Bw[2][2] = {{0, 0}, {0, 0}}, zword[2] = {0, 0};                   // per party: 128 bit registers in two words
    auto getb = [&](int b, int r) -> uint64_t { return ((r < 64 ? Bw[b][0] : Bw[b][1]) >> (r & 63)) & 1ull; };
    auto setb = [&](int b, int r, uint64_t v) {
        const uint64_t m = 1ull << (r & 63), x = (v & 1ull) << (r & 63);
        if (r < 64) Bw[b][0] = (Bw[b][0] & ~m) | x; else Bw[b][1] = (Bw[b][1] & ~m) | x;
    };
    for (int pc = 0; pc < a.n_ins; ++pc) {
        const Ins o = a.ins[pc];
        switch (o.op) {
        case I_B_CONST: setb(0, o.dst, o.imm); setb(1, o.dst, 0); break;
        case I_B_ATOM: setb(0, o.dst, a.bits[0][e] >> o.a); setb(1, o.dst, a.bits[1][e] >> o.a); break;
        case I_B_KAPPA: setb(0, o.dst, kld(a.key[0], a.k.kb, e) >> o.a); setb(1, o.dst, kld(a.key[1], a.k.kb, e) >> o.a); break;
        case I_B_XHAT: setb(0, o.dst, xh >> o.a); setb(1, o.dst, 0); break;
        case I_B_NOT: setb(0, o.dst, getb(0, o.a) ^ 1ull); setb(1, o.dst, getb(1, o.a)); break;
        case I_B_XOR: setb(0, o.dst, getb(0, o.a) ^ getb(0, o.b)); setb(1, o.dst, getb(1, o.a) ^ getb(1, o.b)); break;
        case I_B_ANDPUB: { const uint64_t pub = (xh >> o.b) ^ o.imm; setb(0, o.dst, getb(0, o.a) & pub); setb(1, o.dst, getb(1, o.a) & pub); break; }
        case I_B_OUT: zword[0] |= getb(0, o.a) << o.dst; zword[1] |= getb(1, o.a) << o.dst; break;
        case I_B_AND: {
            uint64_t ta[2], tb[2], tc[2], dm[2], em[2];
#pragma unroll
            for (int b = 0; b < 2; ++b) {
                ta[b] = (kld(a.key[b], a.k.andt, e) >> o.gate) & 1; tb[b] = (kld(a.key[b], a.k.andt + a.k.s8, e) >> o.gate) & 1;
                tc[b] = (kld(a.key[b], a.k.andt + 2 * a.k.s8, e) >> o.gate) & 1;
                dm[b] = getb(b, o.a) ^ ta[b]; em[b] = getb(b, o.b) ^ tb[b];
            }
            const uint64_t dd = dm[0] ^ dm[1], ee = em[0] ^ em[1];
            setb(0, o.dst, (dd & ee) ^ (dd & tb[0]) ^ (ee & ta[0]) ^ tc[0]);
            setb(1, o.dst, (dd & tb[1]) ^ (ee & ta[1]) ^ tc[1]);
            break; }
        case I_A_CONST: A[0][o.dst] = o.imm & mask; A[1][o.dst] = 0; break;
        case I_A_X: A[0][o.dst] = (xh - kld(a.key[0], a.k.rin, e)) & mask; A[1][o.dst] = (0ull - kld(a.key[1], a.k.rin, e)) & mask; break;
        case I_A_COEFF: A[0][o.dst] = a.coeff[0][(size_t)o.a * a.count + e] & mask; A[1][o.dst] = a.coeff[1][(size_t)o.a * a.count + e] & mask; break;
        case I_A_KAPPA: A[0][o.dst] = kld(a.key[0], a.k.ka + (size_t)o.a * a.k.s8, e); A[1][o.dst] = kld(a.key[1], a.k.ka + (size_t)o.a * a.k.s8, e); break;
        case I_A_XHAT_SHR: A[0][o.dst] = o.a >= 64 ? 0ull : xh >> o.a; A[1][o.dst] = 0; break;
        case I_A_ADD: A[0][o.dst] = (A[0][o.a] + A[0][o.b]) & mask; A[1][o.dst] = (A[1][o.a] + A[1][o.b]) & mask; break;
        case I_A_SUB: A[0][o.dst] = (A[0][o.a] - A[0][o.b]) & mask; A[1][o.dst] = (A[1][o.a] - A[1][o.b]) & mask; break;
        case I_A_MULC: A[0][o.dst] = (A[0][o.a] * o.imm) & mask; A[1][o.dst] = (A[1][o.a] * o.imm) & mask; break;
        case I_A_MULXH: A[0][o.dst] = (A[0][o.a] * xh) & mask; A[1][o.dst] = (A[1][o.a] * xh) & mask; break;
        case I_A_OUT:
#pragma unroll
            for (int b = 0; b < 2; ++b) {
                uint64_t v = A[b][o.a];
                if (a.mask_output) v = (v + kld(a.key[b], a.k.rout + (size_t)o.dst * a.k.s8, e)) & mask;
                a.y_out[b][(size_t)o.dst * a.count + e] = v;
            }
            break;
        case I_A_MUL: {
            const size_t to = a.k.beaver + (size_t)o.imm * a.k.s8;
            uint64_t ta[2], tb[2], tc[2], em[2], fm[2];
#pragma unroll
            for (int b = 0; b < 2; ++b) {
                ta[b] = kld(a.key[b], to, e); tb[b] = kld(a.key[b], to + a.k.s8, e); tc[b] = kld(a.key[b], to + 2 * a.k.s8, e);
                em[b] = (A[b][o.a] - ta[b]) & mask; fm[b] = (A[b][o.b] - tb[b]) & mask;
            }
            const uint64_t E = (em[0] + em[1]) & mask, F = (fm[0] + fm[1]) & mask;
            A[0][o.dst] = (E * F + E * tb[0] + F * ta[0] + tc[0]) & mask;
            A[1][o.dst] = (E * tb[1] + F * ta[1] + tc[1]) & mask;
            break; }
        case I_A_MULX: {
            const size_t to = a.k.beaver + (size_t)o.imm * a.k.s8;
            uint64_t tb[2], tc[2], fm[2];
#pragma unroll
            for (int b = 0; b < 2; ++b) { tb[b] = kld(a.key[b], to, e); tc[b] = kld(a.key[b], to + a.k.s8, e); fm[b] = (A[b][o.a] - tb[b]) & mask; }
            const uint64_t F = (fm[0] + fm[1]) & mask;
#pragma unroll
            for (int b = 0; b < 2; ++b) A[b][o.dst] = (xh * A[b][o.a] - F * kld(a.key[b], a.k.rin, e) - tc[b]) & mask;
            break; }
        case I_A_B2A: {
            uint64_t rb[2], ra[2], mm[2];
#pragma unroll
            for (int b = 0; b < 2; ++b) {
                rb[b] = (kld(a.key[b], a.k.b2a_bits, e) >> o.gate) & 1; ra[b] = kld(a.key[b], a.k.b2a_a + (size_t)o.gate * a.k.s8, e);
                mm[b] = getb(b, o.a) ^ rb[b];
            }
            const uint64_t mu = mm[0] ^ mm[1];
            A[0][o.dst] = (mu + ra[0] - 2 * mu * ra[0]) & mask;
            A[1][o.dst] = (ra[1] - 2 * mu * ra[1]) & mask;
            break; }
        case I_B_LSB: setb(0, o.dst, A[0][o.a]); setb(1, o.dst, A[1][o.a]); break;
        case I_B_A2B:
            if (A2B) {
                const int j = (int)o.imm, g = o.gate;
                const uint64_t E = (A[0][o.a] + A[1][o.a] + kld(a.key[0], a.k.a2b_rho + (size_t)g * a.k.s8, e) +
                                    kld(a.key[1], a.k.a2b_rho + (size_t)g * a.k.s8, e)) & mask;
#pragma unroll
                for (int b = 0; b < 2; ++b) {
                    const uint32_t c = bit_tree_eval<false>(tl, a.key[b], a.k.a2b_root[g], a.k.a2b_cw[g], a.k.a2b_vb[g], e, a.k.s16, j,
                                                            E << (64 - j), b, a.k.et);
                    setb(b, o.dst, (b == 0 ? (E >> j) : 0ull) ^ (kld(a.key[b], a.k.a2b_bits, e) >> g) ^ (uint64_t)c);
                }
            }
            break;
        default: break;
        }
    }
    if (a.n_out_b > 0) { a.z_out[0][e] = zword[0]; a.z_out[1][e] = zword[1]; }
    }
}

}  // namespace fsk
