/*
 * oracle/fusefss_oracle.c -- CPU ORACLE.  TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, step-by-step CPU implementation of what the FuseFSS hot path
 * computes (arxiv/paper_2606_09551; citations are /root/reference/PAPER.md
 * lines, "P:<line>").  It shares no code, header, table or helper with the
 * CUDA path under paper_2606_09551_b200/; only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may load it.
 *
 * Two tiers:
 *   Tier A  plaintext semantics  F(x) (Def 4.1) and
 *           G(x) = Phi(F(x), kappa, x, xhat, pub) (Def 4.2).
 *   Tier B  the keyed algorithm, in the paper's order: Protocol 3,
 *           masked rewrites (Lemma 4.3, Lemma E.1, J.3
 *           P:817-843), packed comparison (Def I.1), interval lookup
 *           (Def I.2), online evaluation steps 1-6.
 *
 * The paper treats the DCF, the PRG, the key format and the Beaver/AND/B2A
 * subprotocols as black boxes.  The readings taken here are
 * DESIGN.md section 4 ("KEYFORMAT"); the byte-level key layout and the
 * randomness slot table are "parity unpinned" by the paper (nothing printed to
 * pin them to); everything that has a plain definition -- reconstruction of
 * every share to F(x)/G(x), the DCF truth table, Protocol 3's post-conditions,
 * AES-128 against FIPS-197 -- is pinned in tests/ (-m "not gpu").
 *
 * Variant bit 3 (spec.variant & 8): early-terminated bit trees (dcf_bit_gen_et / dcf_bit_eval_et),
 * pinned by the brute-force truth table at k = 1..12 and by exhaustive reconstruction at n = 8.
 * Variant 1 (spec.variant = 1): the single-key shared-prefix construction -- one DCF key
 * f_{r_k,1} per view width, evaluated point by point from the root (sp_eval); pinned in tests/test_oracle_sp.py.
 *
 * Arithmetic: integers only.  Ring elements are uint64_t with bits >= n zero.
 * 2^n (n = 64) is handled with unsigned __int128, never as a ring element.
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#include <stdio.h>

typedef uint8_t u8;
typedef uint16_t u16;
typedef uint32_t u32;
typedef uint64_t u64;
typedef unsigned __int128 u128;

#define PMAX 8          /* max payload words p                                   */
#define QMAX 4          /* max payload PRG blocks per level, Q = ceil(p/2)       */
#define TMAX 64         /* max atoms (packed in one 64-bit word)                 */
#define MMAX 64         /* max lookup intervals                                  */
#define REGMAX 1024     /* oracle-internal register file (no reuse, SSA)         */
#define OPMAX 4096

/* ------------------------------------------------------------------------- */
/* 1. ring helpers                                                   */
/* ------------------------------------------------------------------------- */
static u64 ring_mask(int n) { return n >= 64 ? ~(u64)0 : (((u64)1 << n) - 1); }
static u64 low_mask(int k) { return ring_mask(k); }

/* ------------------------------------------------------------------------- */
/* 2. AES-128, written from FIPS-197 (sections 4.2, 5.1, 5.2).  Byte oriented. */
/* ------------------------------------------------------------------------- */
static u8 SR[16];                           /* ShiftRows source index, filled from its definition */
static u8 SBOX[256], MUL2[256], MUL3[256];   /* S-box; {02}*x and {03}*x (FIPS-197 4.2.1) */
static int aes_tables_ready = 0;

static u8 gf_mul(u8 a, u8 b)               /* FIPS-197 4.2: multiply mod x^8+x^4+x^3+x+1 */
{
    u8 p = 0;
    for (int i = 0; i < 8; i++) {
        if (b & 1) p ^= a;
        u8 hi = a & 0x80;
        a <<= 1;
        if (hi) a ^= 0x1b;
        b >>= 1;
    }
    return p;
}
static u8 rotl8(u8 x, int s) { return (u8)((x << s) | (x >> (8 - s))); }

static void aes_tables(void)               /* FIPS-197 5.1.1: S-box = affine(inverse) */
{
    if (aes_tables_ready) return;
    for (int x = 0; x < 256; x++) {
        u8 inv = 0;
        if (x) for (int y = 1; y < 256; y++) if (gf_mul((u8)x, (u8)y) == 1) { inv = (u8)y; break; }
        SBOX[x] = inv ^ rotl8(inv, 1) ^ rotl8(inv, 2) ^ rotl8(inv, 3) ^ rotl8(inv, 4) ^ 0x63;
        MUL2[x] = gf_mul((u8)x, 2);
        MUL3[x] = gf_mul((u8)x, 3);
    }
    for (int r = 0; r < 4; r++) for (int c = 0; c < 4; c++) SR[r + 4 * c] = (u8)(r + 4 * ((c + r) % 4));
    aes_tables_ready = 1;
}

typedef struct { u8 rk[11][16]; } aes_ks;

static void aes_expand(const u8 key[16], aes_ks *ks)      /* FIPS-197 5.2, Nk=4, Nr=10 */
{
    aes_tables();
    u8 w[44][4];
    for (int i = 0; i < 4; i++) for (int j = 0; j < 4; j++) w[i][j] = key[4 * i + j];
    u8 rcon = 1;
    for (int i = 4; i < 44; i++) {
        u8 t[4] = { w[i - 1][0], w[i - 1][1], w[i - 1][2], w[i - 1][3] };
        if (i % 4 == 0) {
            u8 t0 = t[0];                                   /* RotWord, SubWord, Rcon */
            t[0] = SBOX[t[1]] ^ rcon; t[1] = SBOX[t[2]]; t[2] = SBOX[t[3]]; t[3] = SBOX[t0];
            rcon = gf_mul(rcon, 2);
        }
        for (int j = 0; j < 4; j++) w[i][j] = w[i - 4][j] ^ t[j];
    }
    for (int r = 0; r < 11; r++) for (int c = 0; c < 4; c++) for (int j = 0; j < 4; j++)
        ks->rk[r][4 * c + j] = w[4 * r + c][j];
}

static void aes_encrypt(const aes_ks *ks, const u8 in[16], u8 out[16])   /* FIPS-197 5.1 */
{
    u8 s[16];                                   /* s[r + 4c] = state row r, column c */
    for (int i = 0; i < 16; i++) s[i] = in[i] ^ ks->rk[0][i];
    for (int round = 1; round <= 10; round++) {
        u8 t[16];
        for (int i = 0; i < 16; i++) t[i] = SBOX[s[i]];                 /* SubBytes  */
        for (int i = 0; i < 16; i++) s[i] = t[SR[i]];                   /* ShiftRows: s[r][c] = t[r][(c+r) mod 4] */
        if (round < 10) {                                               /* MixColumns */
            for (int c = 0; c < 4; c++) {
                u8 a0 = s[4 * c], a1 = s[4 * c + 1], a2 = s[4 * c + 2], a3 = s[4 * c + 3];
                t[4 * c + 0] = MUL2[a0] ^ MUL3[a1] ^ a2 ^ a3;
                t[4 * c + 1] = a0 ^ MUL2[a1] ^ MUL3[a2] ^ a3;
                t[4 * c + 2] = a0 ^ a1 ^ MUL2[a2] ^ MUL3[a3];
                t[4 * c + 3] = MUL3[a0] ^ a1 ^ a2 ^ MUL2[a3];
            }
            memcpy(s, t, 16);
        }
        for (int i = 0; i < 16; i++) s[i] ^= ks->rk[round][i];          /* AddRoundKey */
    }
    memcpy(out, s, 16);
}

void orc_aes128_encrypt(const u8 *key, const u8 *in, u8 *out)
{
    aes_ks ks; aes_expand(key, &ks); aes_encrypt(&ks, in, out);
}

/* ------------------------------------------------------------------------- */
/* 3. PRG.  PRG_i(s, tau) = AES_{K_i}(s ^ tau) ^ (s ^ tau),    */
/*    K_i = bytes (i, 01, 02, .., 0f); tau in {0,1,2} XORed into byte 0.       */
/*    i = 0: child seeds / control bits; i = 1+q: payload block q.             */
/* ------------------------------------------------------------------------- */
static aes_ks PRG_KS[1 + QMAX];
static int prg_ready = 0;
static void prg_init(void)
{
    if (prg_ready) return;
    for (int i = 0; i < 1 + QMAX; i++) {
        u8 key[16];
        for (int j = 0; j < 16; j++) key[j] = (u8)j;
        key[0] = (u8)i;
        aes_expand(key, &PRG_KS[i]);
    }
    prg_ready = 1;
}
static void prg(int i, const u8 s[16], int tau, u8 out[16])
{
    u8 x[16];
    memcpy(x, s, 16);
    x[0] ^= (u8)tau;
    aes_encrypt(&PRG_KS[i], x, out);
    for (int j = 0; j < 16; j++) out[j] ^= x[j];
}
void orc_prg(int i, const u8 *s, int tau, u8 *out) { prg_init(); prg(i, s, tau, out); }

static u64 le64(const u8 *b)
{
    u64 v = 0;
    for (int i = 7; i >= 0; i--) v = (v << 8) | b[i];
    return v;
}
static void put64(u8 *b, u64 v) { for (int i = 0; i < 8; i++) { b[i] = (u8)v; v >>= 8; } }

/* child in direction d: seed (low 2 bits cleared), control bit t = bit 0, Z_2 payload v = bit 1 */
static void child(const u8 s[16], int d, u8 S[16], int *t, int *v)
{
    u8 blk[16];
    prg(0, s, d, blk);
    *t = blk[0] & 1;
    *v = (blk[0] >> 1) & 1;
    memcpy(S, blk, 16);
    S[0] &= 0xFC;
}
/* p ring words for tweak tau (0/1 = direction, 2 = leaf conversion): word w = 64-bit LE chunk w & mask */
static void payload(const u8 s[16], int tau, int p, u64 mask, u64 *W)
{
    int Q = (p + 1) / 2;
    for (int q = 0; q < Q; q++) {
        u8 blk[16];
        prg(1 + q, s, tau, blk);
        if (2 * q < p) W[2 * q] = le64(blk) & mask;
        if (2 * q + 1 < p) W[2 * q + 1] = le64(blk + 8) & mask;
    }
}
static int conv_bit(const u8 s[16])
{
    u8 blk[16];
    prg(0, s, 2, blk);
    return (blk[0] >> 1) & 1;
}

/* ------------------------------------------------------------------------- */
/* 4. DCF (restated from Boyle et al. 2021, cited at P:329-331) */
/*    f_{alpha,beta}(u) = beta if u < alpha else 0, u in [0, 2^k), MSB first.  */
/* ------------------------------------------------------------------------- */
typedef struct { u8 root[16]; u8 cw[64][16]; u64 vbits; } bitkey;   /* root bit0 = final CW bit */
typedef struct { u8 root[16]; u8 scw[64][16]; u64 vcw[64][PMAX]; u64 fin[PMAX]; } veckey;

static void xor16(u8 *d, const u8 *a, const u8 *b) { for (int i = 0; i < 16; i++) d[i] = a[i] ^ b[i]; }

/* payload group Z_2, beta = 1 */
static void dcf_bit_gen(int k, u64 alpha, const u8 r0[16], const u8 r1[16], bitkey *K0, bitkey *K1)
{
    u8 s[2][16];
    memcpy(s[0], r0, 16); memcpy(s[1], r1, 16);
    s[0][0] &= 0xFC; s[1][0] &= 0xFC;
    memset(K0, 0, sizeof *K0); memset(K1, 0, sizeof *K1);
    memcpy(K0->root, s[0], 16); memcpy(K1->root, s[1], 16);
    int t[2] = { 0, 1 };
    int Va = 0;
    u64 vbits = 0;
    for (int i = 0; i < k; i++) {
        int a = (int)((alpha >> (k - 1 - i)) & 1);
        u8 S[2][2][16]; int T[2][2], W[2][2];
        for (int b = 0; b < 2; b++) for (int d = 0; d < 2; d++) child(s[b], d, S[b][d], &T[b][d], &W[b][d]);
        int keep = a, lose = 1 - a;
        u8 sCW[16];
        xor16(sCW, S[0][lose], S[1][lose]);
        int VCW = W[1][lose] ^ W[0][lose] ^ Va ^ (lose == 0 ? 1 : 0);
        Va = Va ^ W[1][keep] ^ W[0][keep] ^ VCW;
        int tCW[2];
        tCW[0] = T[0][0] ^ T[1][0] ^ a ^ 1;
        tCW[1] = T[0][1] ^ T[1][1] ^ a;
        memcpy(K0->cw[i], sCW, 16);
        K0->cw[i][0] |= (u8)(tCW[0] | (tCW[1] << 1));
        vbits |= (u64)VCW << i;
        for (int b = 0; b < 2; b++) {
            u8 ns[16];
            memcpy(ns, S[b][keep], 16);
            if (t[b]) xor16(ns, ns, sCW);
            int nt = T[b][keep] ^ (t[b] & tCW[keep]);
            memcpy(s[b], ns, 16);
            t[b] = nt;
        }
    }
    int fin = conv_bit(s[1]) ^ conv_bit(s[0]) ^ Va;
    K0->vbits = vbits;
    K0->root[0] |= (u8)fin;
    memcpy(K1->cw, K0->cw, sizeof K0->cw);
    K1->vbits = vbits;
    K1->root[0] |= (u8)fin;
}

static int dcf_bit_eval(int b, int k, const bitkey *K, u64 u)
{
    u8 s[16];
    memcpy(s, K->root, 16);
    int fin = s[0] & 1;
    s[0] &= 0xFC;
    int t = b, V = 0;
    for (int i = 0; i < k; i++) {
        int d = (int)((u >> (k - 1 - i)) & 1);
        u8 S[16]; int T, W;
        child(s, d, S, &T, &W);
        V ^= W ^ (t & (int)((K->vbits >> i) & 1));
        if (t) {
            u8 scw[16];
            memcpy(scw, K->cw[i], 16);
            int tcw = (scw[0] >> d) & 1;
            scw[0] &= 0xFC;
            xor16(S, S, scw);
            T ^= tcw;
        }
        memcpy(s, S, 16);
        t = T;
    }
    V ^= conv_bit(s) ^ (t & fin);
    return V;
}

/* Early-terminated bit-DCF (variant bit 3; SURVEY 8(f)-4 "early termination of the GGM tree").
 * A Z_2 payload needs one bit per leaf, a PRG block has 128: the tree is cut nu = max(k-7, 0) levels deep and walks only the
 * top nu input bits u_hi; the leaf seed expands to ONE 128-bit block whose bit u_lo (the remaining lam = min(k,7) input bits)
 * is the leaf's output.  Levels are unchanged (scalar Z_2 contributions W, VCW; all leaves left of alpha_hi output 1 on their
 * whole sub-range, i.e. the level payload is the scalar 1).  Leaf correction block (replaces the one-bit final CW):
 *   L = conv128(s_0) ^ conv128(s_1) ^ X,   X_j = Valpha ^ I[j < alpha_lo],  j = 0..127,   conv128(s) = PRG_0(s, 2),
 * so that on the alpha path (t_0 ^ t_1 = 1) the two leaf blocks differ by X and the output is I[u_lo < alpha_lo], and off the
 * path they cancel.  Bit j of a block = bit (j mod 8) of byte (j div 8).  K->cw[nu] holds L; K->vbits bit i = VCW of level i. */
static int et_levels(int k) { return k > 7 ? k - 7 : 0; }
static void dcf_bit_gen_et(int k, u64 alpha, const u8 r0[16], const u8 r1[16], bitkey *K0, bitkey *K1)
{
    int nu = et_levels(k), lam = k - nu;
    u64 alpha_hi = lam >= 64 ? 0 : alpha >> lam, alpha_lo = alpha & low_mask(lam);
    u8 s[2][16];
    memcpy(s[0], r0, 16); memcpy(s[1], r1, 16);
    s[0][0] &= 0xFC; s[1][0] &= 0xFC;
    memset(K0, 0, sizeof *K0); memset(K1, 0, sizeof *K1);
    memcpy(K0->root, s[0], 16); memcpy(K1->root, s[1], 16);
    int t[2] = { 0, 1 };
    int Va = 0;
    u64 vbits = 0;
    for (int i = 0; i < nu; i++) {                       /* identical to dcf_bit_gen over the nu bits of alpha_hi */
        int a = (int)((alpha_hi >> (nu - 1 - i)) & 1);
        u8 S[2][2][16]; int T[2][2], W[2][2];
        for (int b = 0; b < 2; b++) for (int d = 0; d < 2; d++) child(s[b], d, S[b][d], &T[b][d], &W[b][d]);
        int keep = a, lose = 1 - a;
        u8 sCW[16];
        xor16(sCW, S[0][lose], S[1][lose]);
        int VCW = W[1][lose] ^ W[0][lose] ^ Va ^ (lose == 0 ? 1 : 0);
        Va = Va ^ W[1][keep] ^ W[0][keep] ^ VCW;
        int tCW[2];
        tCW[0] = T[0][0] ^ T[1][0] ^ a ^ 1;
        tCW[1] = T[0][1] ^ T[1][1] ^ a;
        memcpy(K0->cw[i], sCW, 16);
        K0->cw[i][0] |= (u8)(tCW[0] | (tCW[1] << 1));
        vbits |= (u64)VCW << i;
        for (int b = 0; b < 2; b++) {
            u8 ns[16];
            memcpy(ns, S[b][keep], 16);
            if (t[b]) xor16(ns, ns, sCW);
            int nt = T[b][keep] ^ (t[b] & tCW[keep]);
            memcpy(s[b], ns, 16);
            t[b] = nt;
        }
    }
    u8 c0[16], c1[16], L[16];
    prg(0, s[0], 2, c0); prg(0, s[1], 2, c1);
    xor16(L, c0, c1);
    for (int j = 0; j < 128; j++) {
        int xj = Va ^ ((u64)j < alpha_lo ? 1 : 0);
        L[j >> 3] ^= (u8)(xj << (j & 7));
    }
    memcpy(K0->cw[nu], L, 16);
    K0->vbits = vbits;
    memcpy(K1->cw, K0->cw, sizeof K0->cw);
    K1->vbits = vbits;
}
static int dcf_bit_eval_et(int b, int k, const bitkey *K, u64 u)
{
    int nu = et_levels(k), lam = k - nu;
    u64 u_hi = lam >= 64 ? 0 : u >> lam, u_lo = u & low_mask(lam);
    u8 s[16];
    memcpy(s, K->root, 16);
    s[0] &= 0xFC;
    int t = b, V = 0;
    for (int i = 0; i < nu; i++) {
        int d = (int)((u_hi >> (nu - 1 - i)) & 1);
        u8 S[16]; int T, W;
        child(s, d, S, &T, &W);
        V ^= W ^ (t & (int)((K->vbits >> i) & 1));
        if (t) {
            u8 scw[16];
            memcpy(scw, K->cw[i], 16);
            int tcw = (scw[0] >> d) & 1;
            scw[0] &= 0xFC;
            xor16(S, S, scw);
            T ^= tcw;
        }
        memcpy(s, S, 16);
        t = T;
    }
    u8 blk[16];
    prg(0, s, 2, blk);
    if (t) xor16(blk, blk, K->cw[nu]);
    return V ^ ((blk[u_lo >> 3] >> (u_lo & 7)) & 1);
}
void orc_dcf_bit_pair_et(int k, u64 alpha, const u8 *seed0, const u8 *seed1, const u64 *us, int nu_, u8 *out0, u8 *out1)
{
    prg_init();
    bitkey *K0 = malloc(sizeof *K0), *K1 = malloc(sizeof *K1);
    dcf_bit_gen_et(k, alpha, seed0, seed1, K0, K1);
    for (int i = 0; i < nu_; i++) { out0[i] = (u8)dcf_bit_eval_et(0, k, K0, us[i]); out1[i] = (u8)dcf_bit_eval_et(1, k, K1, us[i]); }
    free(K0); free(K1);
}

/* payload group R^p = (Z_{2^n})^p */
static void dcf_vec_gen(int k, int p, u64 mask, u64 alpha, const u64 *beta,
                        const u8 r0[16], const u8 r1[16], veckey *K0, veckey *K1)
{
    u8 s[2][16];
    memcpy(s[0], r0, 16); memcpy(s[1], r1, 16);
    s[0][0] &= 0xFC; s[1][0] &= 0xFC;
    memset(K0, 0, sizeof *K0); memset(K1, 0, sizeof *K1);
    memcpy(K0->root, s[0], 16); memcpy(K1->root, s[1], 16);
    int t[2] = { 0, 1 };
    u64 Va[PMAX] = { 0 };
    for (int i = 0; i < k; i++) {
        int a = (int)((alpha >> (k - 1 - i)) & 1);
        u8 S[2][2][16]; int T[2][2], junk; u64 W[2][2][PMAX];
        for (int b = 0; b < 2; b++) for (int d = 0; d < 2; d++) {
            child(s[b], d, S[b][d], &T[b][d], &junk);
            payload(s[b], d, p, mask, W[b][d]);
        }
        int keep = a, lose = 1 - a;
        u8 sCW[16];
        xor16(sCW, S[0][lose], S[1][lose]);
        u64 VCW[PMAX];
        for (int w = 0; w < p; w++) {
            u64 v = W[1][lose][w] - W[0][lose][w] - Va[w];
            if (lose == 0) v += beta[w];
            if (t[1]) v = (u64)0 - v;
            VCW[w] = v & mask;
            u64 x = Va[w] - W[1][keep][w] + W[0][keep][w];
            x += t[1] ? (u64)0 - VCW[w] : VCW[w];
            Va[w] = x & mask;
            K0->vcw[i][w] = VCW[w];
        }
        int tCW[2];
        tCW[0] = T[0][0] ^ T[1][0] ^ a ^ 1;
        tCW[1] = T[0][1] ^ T[1][1] ^ a;
        memcpy(K0->scw[i], sCW, 16);
        K0->scw[i][0] |= (u8)(tCW[0] | (tCW[1] << 1));
        for (int b = 0; b < 2; b++) {
            u8 ns[16];
            memcpy(ns, S[b][keep], 16);
            if (t[b]) xor16(ns, ns, sCW);
            int nt = T[b][keep] ^ (t[b] & tCW[keep]);
            memcpy(s[b], ns, 16);
            t[b] = nt;
        }
    }
    u64 c0[PMAX], c1[PMAX];
    payload(s[0], 2, p, mask, c0);
    payload(s[1], 2, p, mask, c1);
    for (int w = 0; w < p; w++) {
        u64 v = c1[w] - c0[w] - Va[w];
        if (t[1]) v = (u64)0 - v;
        K0->fin[w] = v & mask;
    }
    memcpy(K1->scw, K0->scw, sizeof K0->scw);
    memcpy(K1->vcw, K0->vcw, sizeof K0->vcw);
    memcpy(K1->fin, K0->fin, sizeof K0->fin);
}

static void dcf_vec_eval(int b, int k, int p, u64 mask, const veckey *K, u64 u, u64 *out)
{
    u8 s[16];
    memcpy(s, K->root, 16);
    s[0] &= 0xFC;
    int t = b;
    u64 V[PMAX] = { 0 };
    for (int i = 0; i < k; i++) {
        int d = (int)((u >> (k - 1 - i)) & 1);
        u8 S[16]; int T, junk; u64 W[PMAX];
        child(s, d, S, &T, &junk);
        payload(s, d, p, mask, W);
        for (int w = 0; w < p; w++) V[w] = (V[w] + W[w] + (t ? K->vcw[i][w] : 0)) & mask;
        if (t) {
            u8 scw[16];
            memcpy(scw, K->scw[i], 16);
            int tcw = (scw[0] >> d) & 1;
            scw[0] &= 0xFC;
            xor16(S, S, scw);
            T ^= tcw;
        }
        memcpy(s, S, 16);
        t = T;
    }
    u64 c[PMAX];
    payload(s, 2, p, mask, c);
    for (int w = 0; w < p; w++) {
        u64 v = V[w] + c[w] + (t ? K->fin[w] : 0);
        if (b) v = (u64)0 - v;
        out[w] = v & mask;
    }
}

/* single-instance entry points for the brute-force pins (tests/test_oracle_dcf.py) */
void orc_dcf_bit_pair(int k, u64 alpha, const u8 *seed0, const u8 *seed1, const u64 *us, int nu, u8 *out0, u8 *out1)
{
    prg_init();
    bitkey *K0 = malloc(sizeof *K0), *K1 = malloc(sizeof *K1);
    dcf_bit_gen(k, alpha, seed0, seed1, K0, K1);
    for (int i = 0; i < nu; i++) { out0[i] = (u8)dcf_bit_eval(0, k, K0, us[i]); out1[i] = (u8)dcf_bit_eval(1, k, K1, us[i]); }
    free(K0); free(K1);
}
void orc_dcf_vec_pair(int k, int n, int p, u64 alpha, const u64 *beta, const u8 *seed0, const u8 *seed1,
                      const u64 *us, int nu, u64 *out0, u64 *out1)
{
    prg_init();
    veckey *K0 = malloc(sizeof *K0), *K1 = malloc(sizeof *K1);
    dcf_vec_gen(k, p, ring_mask(n), alpha, beta, seed0, seed1, K0, K1);
    for (int i = 0; i < nu; i++) {
        dcf_vec_eval(0, k, p, ring_mask(n), K0, us[i], out0 + (size_t)i * p);
        dcf_vec_eval(1, k, p, ring_mask(n), K1, us[i], out1 + (size_t)i * p);
    }
    free(K0); free(K1);
}

/* ------------------------------------------------------------------------- */
/* 5. Operator specification (Def 4.1, App. H)             */
/* ------------------------------------------------------------------------- */
enum { BN_CONST = 0, BN_C = 1, BN_D = 2, BN_MSB = 3, BN_CARRY = 4, BN_NOT = 5, BN_XOR = 6, BN_AND = 7, BN_OR = 8 };
typedef struct { u8 kind, k; u16 lhs, rhs; u8 value_is_2k; u8 pad; u64 value; } orc_bitnode;

enum { KA_R_SHR = 1, KB_R_BIT = 2 };
typedef struct { u8 kind, arg; } orc_kappa;

enum {
    PHI_A_CONST = 1, PHI_A_X, PHI_A_Y, PHI_A_KAPPA, PHI_A_XHAT_SHR, PHI_A_ADD, PHI_A_SUB, PHI_A_MULC,
    PHI_A_MUL, PHI_A_B2A, PHI_A_OUT, PHI_A_AUX,
    PHI_B_CONST = 32, PHI_B_Z, PHI_B_KAPPA, PHI_B_XHAT, PHI_B_NOT, PHI_B_XOR, PHI_B_AND, PHI_B_OR,
    PHI_B_ANDPUB, PHI_B_OUT,
    PHI_B_A2B     /* B[dst] = bit b of the ring element A[a]  (A2B: [x] -> <b>; reading DESIGN 15) */
};
typedef struct { u8 op, dst, a, b; u32 pad; u64 imm; } orc_phi_op;

typedef struct {
    u32 n, frac_bits, m, r, d, p_aux, ell;
    u32 n_nodes, n_kappa_a, n_kappa_b, phi_len, n_out_a, n_out_b, mask_output, variant;
    const u64 *alpha;            /* m-1 interior boundaries (alpha_0 = 0, alpha_m = 2^n implied) */
    const u64 *coeff;            /* [m][r][d+1], high degree first                                */
    const u64 *aux;              /* [m][p_aux]                                                    */
    const orc_bitnode *nodes;
    const u16 *bit_root;         /* [m][ell]                                                      */
    const orc_kappa *kappa_a, *kappa_b;
    const orc_phi_op *phi;
} orc_spec;

/* ---- Tier A: plaintext semantics ---------------------------------------- */
static int plain_node(const orc_spec *S, int id, u64 x, u64 r)
{
    const orc_bitnode *nd = &S->nodes[id];
    int n = (int)S->n;
    u64 mask = ring_mask(n);
    switch (nd->kind) {
    case BN_CONST: return (int)(nd->value & 1);
    case BN_C:     /* C_beta(x) = I[rep(x) < beta], beta in [0, 2^n] */
        if (nd->value_is_2k) return 1;
        return x < nd->value;
    case BN_D:     /* D_{gamma,f}(x) = I[(rep(x) mod 2^f) < gamma] */
        if (nd->value_is_2k) return 1;
        return (x & low_mask(nd->k)) < nd->value;
    case BN_MSB:   /* MSB(x + c) = I[rep(x+c) >= 2^{n-1}] */
        return (int)((((x + nd->value) & mask) >> (n - 1)) & 1);
    case BN_CARRY: /* reading R1: carry out of the low k bits of rep(x) + rep(r) */
        return ((x & low_mask(nd->k)) + (u128)(r & low_mask(nd->k))) >> nd->k ? 1 : 0;
    case BN_NOT: return 1 ^ plain_node(S, nd->lhs, x, r);
    case BN_XOR: return plain_node(S, nd->lhs, x, r) ^ plain_node(S, nd->rhs, x, r);
    case BN_AND: return plain_node(S, nd->lhs, x, r) & plain_node(S, nd->rhs, x, r);
    case BN_OR:  return plain_node(S, nd->lhs, x, r) | plain_node(S, nd->rhs, x, r);
    }
    return 0;
}
static int plain_interval(const orc_spec *S, u64 x)
{
    int i = 0;
    for (u32 j = 0; j + 1 < S->m; j++) if (x >= S->alpha[j]) i = (int)j + 1;
    return i;
}
/* F(x) = (P_i(x), B_i(x)) for the unique i with x in I_i. `r` only feeds BN_CARRY helper bits. */
void orc_plain_F(const orc_spec *S, u64 x, u64 r, u64 *y, u8 *z, u64 *aux_out)
{
    u64 mask = ring_mask((int)S->n);
    int i = plain_interval(S, x);
    for (u32 j = 0; j < S->r; j++) {
        const u64 *c = S->coeff + ((size_t)i * S->r + j) * (S->d + 1);
        u64 acc = 0;
        for (u32 k = 0; k <= S->d; k++) acc = (acc * x + c[k]) & mask;   /* sum_k c_k x^k, high degree first */
        y[j] = acc;
    }
    for (u32 j = 0; j < S->ell; j++) z[j] = (u8)plain_node(S, S->bit_root[(size_t)i * S->ell + j], x, r);
    for (u32 j = 0; j < S->p_aux; j++) aux_out[j] = S->aux[(size_t)i * S->p_aux + j] & mask;
}
static u64 kappa_a_value(const orc_spec *S, int t, u64 r)
{
    const orc_kappa *k = &S->kappa_a[t];
    if (k->kind == KA_R_SHR) return k->arg >= 64 ? 0 : r >> k->arg;
    return 0;
}
static int kappa_b_value(const orc_spec *S, int t, u64 r)
{
    const orc_kappa *k = &S->kappa_b[t];
    if (k->kind == KB_R_BIT) return (int)((r >> k->arg) & 1);
    return 0;
}
/* G(x) = Phi(F(x), kappa(r), x, xhat, pub) on cleartext (Def 4.2) */
void orc_plain_G(const orc_spec *S, u64 x, u64 r, u64 *yo, u8 *zo)
{
    u64 mask = ring_mask((int)S->n);
    u64 y[PMAX], aux[PMAX]; u8 z[64];
    orc_plain_F(S, x, r, y, z, aux);
    if (S->phi_len == 0) {
        for (u32 j = 0; j < S->r; j++) yo[j] = y[j];
        for (u32 j = 0; j < S->ell; j++) zo[j] = z[j];
        return;
    }
    u64 xhat = (x + r) & mask;
    u64 A[256] = { 0 }; u8 B[256] = { 0 };
    for (u32 i = 0; i < S->phi_len; i++) {
        const orc_phi_op *o = &S->phi[i];
        switch (o->op) {
        case PHI_A_CONST: A[o->dst] = o->imm & mask; break;
        case PHI_A_X: A[o->dst] = x; break;
        case PHI_A_Y: A[o->dst] = y[o->a]; break;
        case PHI_A_AUX: A[o->dst] = aux[o->a]; break;
        case PHI_A_KAPPA: A[o->dst] = kappa_a_value(S, o->a, r) & mask; break;
        case PHI_A_XHAT_SHR: A[o->dst] = (o->a >= 64 ? 0 : xhat >> o->a); break;
        case PHI_A_ADD: A[o->dst] = (A[o->a] + A[o->b]) & mask; break;
        case PHI_A_SUB: A[o->dst] = (A[o->a] - A[o->b]) & mask; break;
        case PHI_A_MULC: A[o->dst] = (A[o->a] * o->imm) & mask; break;
        case PHI_A_MUL: A[o->dst] = (A[o->a] * A[o->b]) & mask; break;
        case PHI_A_B2A: A[o->dst] = B[o->a]; break;
        case PHI_A_OUT: yo[o->dst] = A[o->a]; break;
        case PHI_B_CONST: B[o->dst] = (u8)(o->imm & 1); break;
        case PHI_B_Z: B[o->dst] = z[o->a]; break;
        case PHI_B_KAPPA: B[o->dst] = (u8)kappa_b_value(S, o->a, r); break;
        case PHI_B_XHAT: B[o->dst] = (u8)((xhat >> o->a) & 1); break;
        case PHI_B_NOT: B[o->dst] = B[o->a] ^ 1; break;
        case PHI_B_XOR: B[o->dst] = B[o->a] ^ B[o->b]; break;
        case PHI_B_AND: B[o->dst] = B[o->a] & B[o->b]; break;
        case PHI_B_OR: B[o->dst] = B[o->a] | B[o->b]; break;
        case PHI_B_ANDPUB: B[o->dst] = B[o->a] & (u8)(((xhat >> o->b) & 1) ^ (o->imm & 1)); break;
        case PHI_B_OUT: zo[o->dst] = B[o->a]; break;
        case PHI_B_A2B: B[o->dst] = (u8)((A[o->a] >> o->b) & 1); break;
        }
    }
}

/* ------------------------------------------------------------------------- */
/* 6. Spec-level compile (Protocol 3 steps (2)-(4))  */
/* ------------------------------------------------------------------------- */
typedef struct { int k; u64 c; int nbeta; u64 beta[TMAX]; int first_atom; int want_carry; } view_t;
typedef struct { int k; u64 c; int is_theta; u64 beta; int carry_idx; } atom_t;

enum {
    C_B_CONST = 1, C_B_ATOM, C_B_KAPPA, C_B_XHAT, C_B_NOT, C_B_XOR, C_B_AND, C_B_ANDPUB, C_B_OUT,
    C_A_CONST, C_A_X, C_A_COEFF, C_A_KAPPA, C_A_XHAT_SHR, C_A_ADD, C_A_SUB, C_A_MULC, C_A_MUL, C_A_B2A, C_A_OUT,
    C_A_MULXH,    /* variant bit 2: share times the PUBLIC masked input xhat, local (DESIGN 11) */
    C_A_MULX,     /* variant bit 1: product with the gate input x = xhat - r_in, one opening (DESIGN 10) */
    C_B_A2B,      /* bit j >= 1 of a shared ring element: masked opening + a j-bit comparison key (DESIGN 15) */
    C_B_LSB       /* bit 0 of a shared ring element: the XOR of the shares' low bits, local */
};
typedef struct { int op, dst, a, b, idx, round; u64 imm; } cop_t;

typedef struct orc_prog {
    orc_spec S;                       /* deep copy */
    int n, m, M, p, T, has_lut, Q;
    u64 mask;
    int nviews; view_t views[TMAX];
    atom_t atoms[TMAX];
    int n_carry;                      /* theta-atoms; kappa^B = carries ++ user bits */
    int n_kb;                         /* total kappa^B bits */
    int MA, MB, GMIX, rounds;
    int GA2B, a2b_bit[64];            /* A2B nodes with bit index j >= 1 (each: one opened ring element, one j-bit bit-DCF) */
    int nops; cop_t ops[OPMAX];
    int nbreg, nareg;
    int brdy[REGMAX], ardy[REGMAX];
    int n_out_a, n_out_b;
    /* per round message shape */
    int r_nmul[16], r_nbits[16];
    int xmul;                         /* variant bit 1 */
    int xpoly;                        /* variant bit 2: payload = coefficients of P_i(X - r_in), Horner in the public xhat */
    int et;                           /* variant bit 3: bit trees are early-terminated (DESIGN 13) */
    int dense;                        /* variant bit 4: dense-table ("DPF-LUT") lookup by full-domain evaluation (DESIGN 14) */
    int r_narr[16];                   /* ring-element arrays opened per round: 2 per Beaver, 1 per x-product */
    int ma_is_x[64], ma_word[65];     /* per arithmetic gate: kind, first word of its material in the key */
    /* lowering memo */
    int node_reg[4096];
    int calpha_reg[MMAX + 1];
    /* variant 1 (single-key shared-prefix construction): one DCF key per view width,
     * threshold r mod 2^k, evaluated at the public points (xhat + delta) mod 2^k */
    int variant;
    int n_w, wk[8], w_npts[8];        /* widths in first-appearance order; points per width             */
    u64 w_delta[8][2 * TMAX + 2];     /* offsets delta, sorted by signed value                           */
    int atom_w[TMAX], atom_ib[TMAX], atom_ia[TMAX];   /* per atom: width, point of (c), point of (c - beta) */
    int alpha_atom[MMAX];             /* atom index of the boundary comparison C_{alpha_i}, i = 1..m-1   */
} orc_prog;

static int find_view(orc_prog *P, int k, u64 c)
{
    for (int v = 0; v < P->nviews; v++) if (P->views[v].k == k && P->views[v].c == c) return v;
    P->views[P->nviews].k = k; P->views[P->nviews].c = c; P->views[P->nviews].nbeta = 0;
    P->views[P->nviews].want_carry = 0;
    return P->nviews++;
}
static void add_pred(orc_prog *P, int k, u64 c, u64 beta)
{
    int v = find_view(P, k, c);
    for (int j = 0; j < P->views[v].nbeta; j++) if (P->views[v].beta[j] == beta) return;
    P->views[v].beta[P->views[v].nbeta++] = beta;
}
static int theta_atom(const orc_prog *P, int k, u64 c, u64 beta)
{
    for (int t = 0; t < P->T; t++)
        if (P->atoms[t].is_theta && P->atoms[t].k == k && P->atoms[t].c == c && P->atoms[t].beta == beta) return t;
    return -1;
}
static int r_atom(const orc_prog *P, int k, u64 c)
{
    for (int t = 0; t < P->T; t++) if (!P->atoms[t].is_theta && P->atoms[t].k == k && P->atoms[t].c == c) return t;
    return -1;
}

static int emit(orc_prog *P, int op, int dst, int a, int b, u64 imm)
{
    cop_t *o = &P->ops[P->nops];
    o->op = op; o->dst = dst; o->a = a; o->b = b; o->imm = imm; o->idx = -1; o->round = -1;
    return P->nops++;
}
static int newb(orc_prog *P, int rdy) { P->brdy[P->nbreg] = rdy; return P->nbreg++; }
static int newa(orc_prog *P, int rdy) { P->ardy[P->nareg] = rdy; return P->nareg++; }
static int imax(int a, int b) { return a > b ? a : b; }

static int e_bconst(orc_prog *P, int v) { int d = newb(P, 0); emit(P, C_B_CONST, d, 0, 0, (u64)v); return d; }
static int e_bxor(orc_prog *P, int a, int b) { int d = newb(P, imax(P->brdy[a], P->brdy[b])); emit(P, C_B_XOR, d, a, b, 0); return d; }
static int e_bnot(orc_prog *P, int a) { int d = newb(P, P->brdy[a]); emit(P, C_B_NOT, d, a, 0, 0); return d; }
static int e_band(orc_prog *P, int a, int b)
{
    int rd = imax(P->brdy[a], P->brdy[b]);
    int d = newb(P, rd + 1);
    int i = emit(P, C_B_AND, d, a, b, 0);
    P->ops[i].idx = P->MB++; P->ops[i].round = rd;
    return d;
}
/* masked rewrite of a primitive predicate I[view_{k,c}(x) < beta]:
 * Lemma 4.3 (restored from the proof P:807-815 and App. N) / Lemma E.1:
 *   = A_theta xor A_r xor w,  w = I[r_k + beta >= 2^k] kept secret-shared (kappa^B). */
static int e_pred(orc_prog *P, int k, u64 c, u64 beta)
{
    int at = theta_atom(P, k, c, beta), ar = r_atom(P, k, c);
    if (P->variant) { int r0 = newb(P, 0); emit(P, C_B_ATOM, r0, at, 0, 0); return r0; }   /* DESIGN 9: no carry, no r-atom */
    int r1 = newb(P, 0); emit(P, C_B_ATOM, r1, at, 0, 0);
    int r2 = newb(P, 0); emit(P, C_B_ATOM, r2, ar, 0, 0);
    int r3 = newb(P, 0); emit(P, C_B_KAPPA, r3, P->atoms[at].carry_idx, 0, 0);
    return e_bxor(P, e_bxor(P, r1, r2), r3);
}
static int lower_node(orc_prog *P, int id)
{
    if (P->node_reg[id] >= 0) return P->node_reg[id];
    const orc_bitnode *nd = &P->S.nodes[id];
    int n = P->n, reg = -1;
    switch (nd->kind) {
    case BN_CONST: reg = e_bconst(P, (int)(nd->value & 1)); break;
    case BN_C:     /* sentinels C_0 = 0, C_N = 1 */
        if (nd->value_is_2k) reg = e_bconst(P, 1);
        else if (nd->value == 0) reg = e_bconst(P, 0);
        else reg = e_pred(P, n, 0, nd->value);
        break;
    case BN_D:     /* sentinels D_{0,f} = 0, D_{2^f,f} = 1 */
        if (nd->value_is_2k) reg = e_bconst(P, 1);
        else if (nd->value == 0) reg = e_bconst(P, 0);
        else reg = e_pred(P, nd->k, 0, nd->value);
        break;
    case BN_MSB:   /* MSB(x+c) = not I[view_{n,c}(x) < 2^{n-1}] */
        reg = e_bnot(P, e_pred(P, n, nd->value & P->mask, (u64)1 << (n - 1)));
        break;
    case BN_CARRY: { int d = newb(P, 0); emit(P, C_B_ATOM, d, r_atom(P, nd->k, 0), 0, 0); reg = d; break; }
    case BN_NOT: reg = e_bnot(P, lower_node(P, nd->lhs)); break;
    case BN_XOR: { int a = lower_node(P, nd->lhs), b = lower_node(P, nd->rhs); reg = e_bxor(P, a, b); break; }
    case BN_AND: { int a = lower_node(P, nd->lhs), b = lower_node(P, nd->rhs); reg = e_band(P, a, b); break; }
    case BN_OR:  { int a = lower_node(P, nd->lhs), b = lower_node(P, nd->rhs);      /* a|b = not(not a & not b) */
                   reg = e_bnot(P, e_band(P, e_bnot(P, a), e_bnot(P, b))); break; }
    }
    P->node_reg[id] = reg;
    return reg;
}
/* C_{alpha_i}(x) for the interval indicators of Lemma D.1; alpha_0 = 0, alpha_m = 2^n sentinels */
static int lower_calpha(orc_prog *P, int i)
{
    if (P->calpha_reg[i] >= 0) return P->calpha_reg[i];
    int reg;
    if (i == 0) reg = e_bconst(P, 0);
    else if (i == P->m) reg = e_bconst(P, 1);
    else reg = e_pred(P, P->n, 0, P->S.alpha[i - 1]);
    P->calpha_reg[i] = reg;
    return reg;
}
static int bit_is_uniform(const orc_spec *S, u32 j)
{
    for (u32 i = 1; i < S->m; i++) if (S->bit_root[(size_t)i * S->ell + j] != S->bit_root[j]) return 0;
    return 1;
}

static void *dup_mem(const void *src, size_t bytes)
{
    void *d = malloc(bytes ? bytes : 1);
    if (bytes) memcpy(d, src, bytes);
    return d;
}

void orc_destroy(orc_prog *P)
{
    if (!P) return;
    free((void *)P->S.alpha); free((void *)P->S.coeff); free((void *)P->S.aux); free((void *)P->S.nodes);
    free((void *)P->S.bit_root); free((void *)P->S.kappa_a); free((void *)P->S.kappa_b); free((void *)P->S.phi);
    free(P);
}

/* variant 1: evaluation points.  For a predicate atom (k, c, beta): I[view_{k,c}(x) < beta] = e - b + a with
 * h = (xhat + c) mod 2^k, e = I[h < beta] public, b = I[h < r_k], a = I[(h - beta) mod 2^k < r_k]  (checked
 * exhaustively in tests/test_oracle_sp.py); b and a are the ONE DCF f_{r_k,1} at the offsets c and c - beta. */
static int sp_point(orc_prog *P, int w, u64 delta)
{
    for (int j = 0; j < P->w_npts[w]; j++) if (P->w_delta[w][j] == delta) return j;
    P->w_delta[w][P->w_npts[w]] = delta;
    return P->w_npts[w]++;
}
static int sp_points(orc_prog *P)
{
    P->n_w = 0;
    for (int t = 0; t < P->T; t++) {                     /* widths in first-appearance order */
        int w = -1;
        for (int i = 0; i < P->n_w; i++) if (P->wk[i] == P->atoms[t].k) w = i;
        if (w < 0) { if (P->n_w >= 8) return -1; w = P->n_w++; P->wk[w] = P->atoms[t].k; P->w_npts[w] = 0; }
        P->atom_w[t] = w;
    }
    for (int pass = 0; pass < 2; pass++) {               /* pass 0 collects, then sort, pass 1 resolves indices */
        for (int t = 0; t < P->T; t++) {
            const atom_t *a = &P->atoms[t];
            int w = P->atom_w[t];
            u64 km = low_mask(a->k);
            P->atom_ib[t] = sp_point(P, w, a->c & km);
            P->atom_ia[t] = a->is_theta ? sp_point(P, w, (a->c - a->beta) & km) : -1;
        }
        if (pass == 0) for (int w = 0; w < P->n_w; w++) {    /* ascending as signed k-bit values */
            int k = P->wk[w]; u64 half = (u64)1 << (k - 1);
            for (int i = 1; i < P->w_npts[w]; i++) {
                u64 v = P->w_delta[w][i]; int j = i;
                while (j > 0 && ((P->w_delta[w][j - 1] ^ half) > (v ^ half))) { P->w_delta[w][j] = P->w_delta[w][j - 1]; j--; }
                P->w_delta[w][j] = v;
            }
        }
    }
    for (int i = 1; i < P->m; i++) P->alpha_atom[i] = P->has_lut ? theta_atom(P, P->n, 0, P->S.alpha[i - 1]) : -1;
    return 0;
}

orc_prog *orc_compile(const orc_spec *S0)
{
    prg_init();
    const orc_spec *S = S0;
    if (S->n < 1 || S->n > 64 || S->m < 1 || S->m >= MMAX) return NULL;
    int p = (int)(S->r * (S->d + 1) + S->p_aux);
    if (p > PMAX) return NULL;
    for (u32 i = 0; i + 1 < S->m; i++) {            /* well-formedness: strictly increasing in (0, 2^n) */
        u64 a = S->alpha[i];
        if (a == 0 || (a & ~ring_mask((int)S->n))) return NULL;
        if (i && a <= S->alpha[i - 1]) return NULL;
    }
    /* well-formedness of the rest of the descriptor ("boundaries, polynomials, constants and gates must be well formed") */
    for (u32 i = 0; i < S->n_nodes; i++) {
        const orc_bitnode *nd = &S->nodes[i];
        if (nd->kind > BN_OR) return NULL;
        if ((nd->kind == BN_D || nd->kind == BN_CARRY) && (nd->k < 1 || nd->k > S->n)) return NULL;
        if (nd->kind == BN_C && !nd->value_is_2k && nd->value > ring_mask((int)S->n)) return NULL;      /* beta in [0, 2^n] */
        if (nd->kind == BN_D && !nd->value_is_2k && nd->value > low_mask(nd->k)) return NULL;          /* gamma in [0, 2^k] */
        if (nd->kind >= BN_NOT && nd->lhs >= i) return NULL;                                           /* operands precede (DAG) */
        if (nd->kind >= BN_XOR && nd->rhs >= i) return NULL;
    }
    for (u32 i = 0; i < S->m * S->ell; i++) if (S->bit_root[i] >= S->n_nodes) return NULL;
    if (S->n_kappa_a > 8 || S->n_kappa_b > 64) return NULL;
    for (u32 i = 0; i < S->n_kappa_a; i++) if (S->kappa_a[i].kind != KA_R_SHR || S->kappa_a[i].arg > 63) return NULL;
    for (u32 i = 0; i < S->n_kappa_b; i++) if (S->kappa_b[i].kind != KB_R_BIT || S->kappa_b[i].arg >= S->n) return NULL;
    if (S->phi_len) {
        int seen_a[256] = { 0 }, seen_b[256] = { 0 };
        for (u32 i = 0; i < S->phi_len; i++) {
            const orc_phi_op *o = &S->phi[i];
            if ((o->op == PHI_B_XHAT && o->a >= S->n) || (o->op == PHI_B_ANDPUB && o->b >= S->n)) return NULL;   /* public bit index < n */
            if (o->op == PHI_A_XHAT_SHR && o->a > 64) return NULL;
            if (o->op == PHI_A_OUT) seen_a[o->dst]++;
            if (o->op == PHI_B_OUT) seen_b[o->dst]++;
        }
        for (u32 j = 0; j < 256; j++) {                       /* every declared output is written exactly once */
            if (seen_a[j] != (j < S->n_out_a)) return NULL;
            if (seen_b[j] != (j < S->n_out_b)) return NULL;
        }
    }
    orc_prog *P = calloc(1, sizeof *P);
    P->S = *S;
    P->S.alpha = dup_mem(S->alpha, sizeof(u64) * (S->m - 1));
    P->S.coeff = dup_mem(S->coeff, sizeof(u64) * S->m * S->r * (S->d + 1));
    P->S.aux = dup_mem(S->aux, sizeof(u64) * S->m * S->p_aux);
    P->S.nodes = dup_mem(S->nodes, sizeof(orc_bitnode) * S->n_nodes);
    P->S.bit_root = dup_mem(S->bit_root, sizeof(u16) * S->m * S->ell);
    P->S.kappa_a = dup_mem(S->kappa_a, sizeof(orc_kappa) * S->n_kappa_a);
    P->S.kappa_b = dup_mem(S->kappa_b, sizeof(orc_kappa) * S->n_kappa_b);
    P->S.phi = dup_mem(S->phi, sizeof(orc_phi_op) * S->phi_len);
    S = &P->S;
    P->n = (int)S->n; P->m = (int)S->m; P->mask = ring_mask(P->n); P->p = p; P->Q = (p + 1) / 2;
    /* M = min(m+1, 2^n)  (Protocol 3 line 2) */
    u128 N = (u128)1 << P->n;
    P->M = ((u128)(P->m + 1) < N) ? P->m + 1 : (int)N;
    P->has_lut = P->m > 1;                               /* single interval: lookup omitted */
    P->variant = (int)(S->variant & 1);
    P->xmul = (int)((S->variant >> 1) & 1);
    P->xpoly = (int)((S->variant >> 2) & 1) && S->d >= 1 && P->m > 1;
    P->et = (int)((S->variant >> 3) & 1);
    P->dense = (int)((S->variant >> 4) & 1);
    if (P->dense && (!P->variant || P->xpoly || P->n > 16)) { orc_destroy(P); return NULL; }   /* needs the single key, n <= 16 */
    if (P->variant) P->M = P->m;                         /* no translated partition, hence no wrap/dummy split */
    for (int i = 0; i < 4096; i++) P->node_reg[i] = -1;
    for (int i = 0; i <= MMAX; i++) P->calpha_reg[i] = -1;

    /* (4) fixed predicate query list: primitive nodes in descriptor (node-array) order, then the
     *     boundary comparisons C_{alpha_i}, i = 1..m-1, iff some output bit is piecewise (Lemma D.2). */
    for (u32 id = 0; id < S->n_nodes; id++) {
        const orc_bitnode *nd = &S->nodes[id];
        if (nd->kind == BN_C && !nd->value_is_2k && nd->value != 0) add_pred(P, P->n, 0, nd->value);
        if (nd->kind == BN_D && !nd->value_is_2k && nd->value != 0) add_pred(P, nd->k, 0, nd->value);
        if (nd->kind == BN_MSB) add_pred(P, P->n, nd->value & P->mask, (u64)1 << (P->n - 1));
        if (nd->kind == BN_CARRY) P->views[find_view(P, nd->k, 0)].want_carry = 1;
    }
    int piecewise = 0;
    for (u32 j = 0; j < S->ell; j++) if (!bit_is_uniform(S, j)) piecewise = 1;
    if (piecewise || ((S->variant & 1) && P->m > 1)) for (int i = 1; i < P->m; i++) add_pred(P, P->n, 0, S->alpha[i - 1]);
    /* flatten: per view, the r-atom then one theta-atom per distinct beta */
    P->T = 0; P->n_carry = 0;
    for (int v = 0; v < P->nviews; v++) {
        view_t *V = &P->views[v];
        V->first_atom = P->T;
        if (P->T + 1 + V->nbeta > TMAX) { orc_destroy(P); return NULL; }
        atom_t *a;
        if (!(S->variant & 1) || V->want_carry) {              /* variant 1 keeps the r-atom only where a CARRY node reads it */
            a = &P->atoms[P->T++];
            a->k = V->k; a->c = V->c; a->is_theta = 0; a->beta = 0; a->carry_idx = -1;
        }
        for (int j = 0; j < V->nbeta; j++) {
            a = &P->atoms[P->T++];
            a->k = V->k; a->c = V->c; a->is_theta = 1; a->beta = V->beta[j];
            a->carry_idx = (S->variant & 1) ? -1 : P->n_carry++;
        }
    }
    P->n_kb = P->n_carry + (int)S->n_kappa_b;
    if ((S->variant & 1) && sp_points(P) < 0) { orc_destroy(P); return NULL; }

    /* program: Horner (step-major), Boolean circuit (bit-major), then Phi */
    int xreg = newa(P, 0); emit(P, C_A_X, xreg, 0, 0, 0);
    int yreg[PMAX], auxreg[PMAX], zreg[64];
    int creg[PMAX];
    for (int w = 0; w < p; w++) {
        creg[w] = newa(P, 0);
        if (P->has_lut) emit(P, C_A_COEFF, creg[w], w, 0, 0);
        else {                                           /* m = 1: coefficients are public descriptor constants */
            u64 v = (w < (int)(S->r * (S->d + 1))) ? S->coeff[w] : S->aux[w - S->r * (S->d + 1)];
            emit(P, C_A_CONST, creg[w], 0, 0, v & P->mask);
        }
    }
    for (u32 j = 0; j < S->r; j++) yreg[j] = creg[j * (S->d + 1)];
    for (u32 k = 1; k <= S->d; k++)                      /* Horner: acc = acc*x + c_k, one round per step */
        for (u32 j = 0; j < S->r; j++) {
            if (P->xpoly) {                              /* y = (..(c'_d xhat + c'_{d-1}) xhat ..) + c'_0: no interaction (DESIGN 11) */
                int pr = newa(P, P->ardy[yreg[j]]);
                emit(P, C_A_MULXH, pr, yreg[j], 0, 0);
                int sm = newa(P, P->ardy[yreg[j]]);
                emit(P, C_A_ADD, sm, pr, creg[j * (S->d + 1) + k], 0);
                yreg[j] = sm;
                continue;
            }
            int rd = imax(P->ardy[yreg[j]], P->ardy[xreg]);
            int prod = newa(P, rd + 1);
            int i = emit(P, P->xmul ? C_A_MULX : C_A_MUL, prod, yreg[j], xreg, 0);
            P->ops[i].idx = P->MA++; P->ops[i].round = rd;
            int sum = newa(P, rd + 1);
            emit(P, C_A_ADD, sum, prod, creg[j * (S->d + 1) + k], 0);
            yreg[j] = sum;
        }
    for (u32 j = 0; j < S->p_aux; j++) auxreg[j] = creg[S->r * (S->d + 1) + j];
    for (u32 j = 0; j < S->ell; j++) {
        if (bit_is_uniform(S, j)) zreg[j] = lower_node(P, S->bit_root[j]);
        else {                                           /* B^{(j)} = XOR_i (J_i and B_i^{(j)})  (Lemma D.2) */
            int acc = -1;
            for (int i = 0; i < P->m; i++) {
                int J = e_bxor(P, lower_calpha(P, i + 1), lower_calpha(P, i));
                int Bi = lower_node(P, S->bit_root[(size_t)i * S->ell + j]);
                int term = e_band(P, J, Bi);
                acc = acc < 0 ? term : e_bxor(P, acc, term);
            }
            zreg[j] = acc;
        }
    }
    if (S->phi_len == 0) {
        P->n_out_a = (int)S->r; P->n_out_b = (int)S->ell;
        for (u32 j = 0; j < S->r; j++) emit(P, C_A_OUT, (int)j, yreg[j], 0, 0);
        for (u32 j = 0; j < S->ell; j++) emit(P, C_B_OUT, (int)j, zreg[j], 0, 0);
    } else {
        P->n_out_a = (int)S->n_out_a; P->n_out_b = (int)S->n_out_b;
        int ua[256], ub[256];
        for (int i = 0; i < 256; i++) ua[i] = ub[i] = -1;
        for (u32 i = 0; i < S->phi_len; i++) {
            const orc_phi_op *o = &S->phi[i];
            int d, k;
            switch (o->op) {
            case PHI_A_CONST: d = newa(P, 0); emit(P, C_A_CONST, d, 0, 0, o->imm & P->mask); ua[o->dst] = d; break;
            case PHI_A_X: ua[o->dst] = xreg; break;
            case PHI_A_Y: ua[o->dst] = yreg[o->a]; break;
            case PHI_A_AUX: ua[o->dst] = auxreg[o->a]; break;
            case PHI_A_KAPPA: d = newa(P, 0); emit(P, C_A_KAPPA, d, o->a, 0, 0); ua[o->dst] = d; break;
            case PHI_A_XHAT_SHR: d = newa(P, 0); emit(P, C_A_XHAT_SHR, d, o->a, 0, 0); ua[o->dst] = d; break;
            case PHI_A_ADD: d = newa(P, imax(P->ardy[ua[o->a]], P->ardy[ua[o->b]])); emit(P, C_A_ADD, d, ua[o->a], ua[o->b], 0); ua[o->dst] = d; break;
            case PHI_A_SUB: d = newa(P, imax(P->ardy[ua[o->a]], P->ardy[ua[o->b]])); emit(P, C_A_SUB, d, ua[o->a], ua[o->b], 0); ua[o->dst] = d; break;
            case PHI_A_MULC: d = newa(P, P->ardy[ua[o->a]]); emit(P, C_A_MULC, d, ua[o->a], 0, o->imm); ua[o->dst] = d; break;
            case PHI_A_MUL: {
                int rd = imax(P->ardy[ua[o->a]], P->ardy[ua[o->b]]);
                int ax = ua[o->a] == xreg, bx = ua[o->b] == xreg;
                d = newa(P, rd + 1);
                if (P->xmul && ax != bx) k = emit(P, C_A_MULX, d, ax ? ua[o->b] : ua[o->a], xreg, 0);
                else k = emit(P, C_A_MUL, d, ua[o->a], ua[o->b], 0);
                P->ops[k].idx = P->MA++; P->ops[k].round = rd; ua[o->dst] = d; break; }
            case PHI_A_B2A: {
                int rd = P->brdy[ub[o->a]];
                d = newa(P, rd + 1); k = emit(P, C_A_B2A, d, ub[o->a], 0, 0);
                P->ops[k].idx = P->GMIX++; P->ops[k].round = rd; ua[o->dst] = d; break; }
            case PHI_A_OUT: emit(P, C_A_OUT, o->dst, ua[o->a], 0, 0); break;
            case PHI_B_CONST: ub[o->dst] = e_bconst(P, (int)(o->imm & 1)); break;
            case PHI_B_Z: ub[o->dst] = zreg[o->a]; break;
            case PHI_B_KAPPA: d = newb(P, 0); emit(P, C_B_KAPPA, d, P->n_carry + o->a, 0, 0); ub[o->dst] = d; break;
            case PHI_B_XHAT: d = newb(P, 0); emit(P, C_B_XHAT, d, o->a, 0, 0); ub[o->dst] = d; break;
            case PHI_B_NOT: ub[o->dst] = e_bnot(P, ub[o->a]); break;
            case PHI_B_XOR: ub[o->dst] = e_bxor(P, ub[o->a], ub[o->b]); break;
            case PHI_B_AND: ub[o->dst] = e_band(P, ub[o->a], ub[o->b]); break;
            case PHI_B_OR: ub[o->dst] = e_bnot(P, e_band(P, e_bnot(P, ub[o->a]), e_bnot(P, ub[o->b]))); break;
            case PHI_B_ANDPUB: d = newb(P, P->brdy[ub[o->a]]); emit(P, C_B_ANDPUB, d, ub[o->a], o->b, o->imm & 1); ub[o->dst] = d; break;
            case PHI_B_OUT: emit(P, C_B_OUT, o->dst, ub[o->a], 0, 0); break;
            case PHI_B_A2B: {
                if (o->b >= S->n || ua[o->a] < 0) { orc_destroy(P); return NULL; }
                if (o->b == 0) { d = newb(P, P->ardy[ua[o->a]]); emit(P, C_B_LSB, d, ua[o->a], 0, 0); ub[o->dst] = d; break; }
                int rd = P->ardy[ua[o->a]];
                if (P->GA2B >= 8) { orc_destroy(P); return NULL; }
                d = newb(P, rd + 1); k = emit(P, C_B_A2B, d, ua[o->a], 0, (u64)o->b);
                P->a2b_bit[P->GA2B] = o->b; P->ops[k].idx = P->GA2B++; P->ops[k].round = rd; ub[o->dst] = d; break; }
            default: orc_destroy(P); return NULL;
            }
        }
    }
    P->rounds = 0;
    for (int i = 0; i < P->nops; i++) if (P->ops[i].round >= 0) P->rounds = imax(P->rounds, P->ops[i].round + 1);
    if (P->rounds > 16 || P->MB > 64 || P->GMIX > 64 || P->MA > 64) { orc_destroy(P); return NULL; }
    for (int i = 0; i < P->nops; i++) {
        cop_t *o = &P->ops[i];
        if (o->round < 0) continue;
        if (o->op == C_A_MUL) { P->r_nmul[o->round]++; P->r_narr[o->round] += 2; P->ma_is_x[o->idx] = 0; }
        if (o->op == C_A_MULX) { P->r_nmul[o->round]++; P->r_narr[o->round] += 1; P->ma_is_x[o->idx] = 1; }
        if (o->op == C_B_AND) P->r_nbits[o->round] += 2;
        if (o->op == C_A_B2A) P->r_nbits[o->round] += 1;
        if (o->op == C_B_A2B) P->r_narr[o->round] += 1;
    }
    /* a round's opened bits travel in ONE 64-bit word per element (message layout, DESIGN 4.6): more than 64 of them (e.g. 33 AND
     * gates in one round) is over the format's limit -- reject instead of shifting past the word */
    for (int q = 0; q < P->rounds; q++) if (P->r_nbits[q] > 64) { orc_destroy(P); return NULL; }
    P->ma_word[0] = 0;
    for (int i = 0; i < P->MA; i++) P->ma_word[i + 1] = P->ma_word[i] + (P->ma_is_x[i] ? 2 : 3);
    return P;
}

/* L_shape: out = T, M, p, M_A, M_B, G_mix, rounds, n_out_a, n_out_b, has_lut, n_kb ; ks[t] = k_t */
void orc_shape(const orc_prog *P, int *out, int *ks)
{
    out[0] = P->T; out[1] = P->M; out[2] = P->p; out[3] = P->MA; out[4] = P->MB; out[5] = P->GMIX + P->GA2B;     /* G_mix = mixed-domain conversions, B2A and A2B */
    out[6] = P->rounds; out[7] = P->n_out_a; out[8] = P->n_out_b; out[9] = P->has_lut; out[10] = P->n_kb;
    for (int t = 0; t < P->T; t++) ks[t] = P->atoms[t].k;
}
/* atom description for tests: k, c, is_theta, beta */
void orc_atom(const orc_prog *P, int t, u64 *out)
{
    out[0] = (u64)P->atoms[t].k; out[1] = P->atoms[t].c; out[2] = (u64)P->atoms[t].is_theta; out[3] = P->atoms[t].beta;
}

/* variant bit 2 (DESIGN 11): coefficient of X^j of P(X - r), P = sum_k c_k X^k:
 *   c'_j = sum_{k >= j} c_k C(k, j) (-r)^{k-j}   (binomial theorem), so that P(x) = sum_j c'_j xhat^j with xhat = x + r. */
static u64 binom(int k, int j)
{
    u64 v = 1;
    for (int i = 1; i <= j; i++) v = v * (u64)(k - j + i) / (u64)i;
    return v;
}
static u64 shifted_coeff(const orc_spec *S, int i, int q, int j, u64 r, u64 mask)
{
    int d = (int)S->d;
    const u64 *c = S->coeff + ((size_t)i * S->r + q) * (d + 1);           /* high degree first: c_k = c[d - k] */
    u64 acc = 0;
    for (int k = j; k <= d; k++) {
        u64 pw = 1;
        for (int t = 0; t < k - j; t++) pw = (pw * ((u64)0 - r)) & mask;
        acc = (acc + c[d - k] * binom(k, j) * pw) & mask;
    }
    return acc;
}

/* ------------------------------------------------------------------------- */
/* 7. Protocol 3 step (1), exactly as written                      */
/* ------------------------------------------------------------------------- */
/* B has M+1 entries (B[M] = 2^n as u128), ord has M entries. */
static void protocol3(int n, int m, const u64 *alpha_interior, u64 r, u128 *B, int *ord, int *M_out)
{
    u128 N = (u128)1 << n;
    int M = ((u128)(m + 1) < N) ? m + 1 : (int)N;                       /* line 2 */
    u64 s[MMAX]; int pi[MMAX];
    for (int i = 0; i < m; i++) {                                       /* lines 5-7 */
        u128 a = (i == 0) ? 0 : alpha_interior[i - 1];
        s[i] = (u64)((a + r) % N);
        pi[i] = i;
    }
    for (int i = 1; i < m; i++) {                                       /* line 8: sort, pi = permutation */
        int j = i;
        while (j > 0 && s[pi[j - 1]] > s[pi[j]]) { int t = pi[j]; pi[j] = pi[j - 1]; pi[j - 1] = t; j--; }
    }
    u64 beta[MMAX];
    for (int j = 0; j < m; j++) beta[j] = s[pi[j]];                     /* line 9 */
    int len;
    if (beta[0] == 0) {                                                 /* line 10 */
        B[0] = 0;
        for (int j = 1; j < m; j++) B[j] = beta[j];
        B[m] = N;
        for (int j = 0; j < m; j++) ord[j] = pi[j];
        len = m;
        if ((u128)m < N) {                                              /* lines 12-18: dummy split */
            int js = 0;
            while (B[js + 1] - B[js] < 2) js++;
            u128 delta = B[js] + 1;
            for (int j = len; j > js; j--) B[j + 1] = B[j];
            B[js + 1] = delta;
            for (int j = len - 1; j > js; j--) ord[j + 1] = ord[j];
            ord[js + 1] = ord[js];
            len = m + 1;
        }
    } else {                                                            /* line 19: wrap split at 0 */
        B[0] = 0;
        for (int j = 0; j < m; j++) B[j + 1] = beta[j];
        B[m + 1] = N;
        ord[0] = pi[m - 1];
        for (int j = 0; j < m; j++) ord[j + 1] = pi[j];
        len = m + 1;
    }
    (void)len;
    *M_out = M;
}
/* test entry: B_out[M+1] truncated to 64 bits (B[M] = 2^n reads 0 when n = 64) */
void orc_protocol3(int n, int m, const u64 *alpha_interior, u64 r, u64 *B_out, int *ord_out, int *M_out)
{
    u128 B[MMAX + 2]; int M;
    protocol3(n, m, alpha_interior, r, B, ord_out, &M);
    for (int j = 0; j <= M; j++) B_out[j] = (u64)B[j];
    *M_out = M;
}

/* ------------------------------------------------------------------------- */
/* 8. Key layout: SoA over the chunk's elements, every array   */
/*    padded to a multiple of 256 bytes.  Depends on (program, count) only     */
/*    -- the testable form of Prop. I.3.                               */
/* ------------------------------------------------------------------------- */
typedef struct {
    size_t s16, s8;
    size_t bt_root[TMAX], bt_cw[TMAX], bt_vb[TMAX];
    size_t lut_c, vt_root[MMAX], vt_lvl[MMAX], vt_fin[MMAX], lvl_stride;
    size_t rin, rout, ka, rpow, kb, beaver, andt, b2a_bits, b2a_a, total;
    size_t a2b_rho, a2b_bits, a2b_root[8], a2b_cw[8], a2b_vb[8];
} layout_t;
static size_t rup256(size_t x) { return (x + 255) & ~(size_t)255; }
/* 16-byte correction arrays of a bit tree on k bits: k levels, or (early termination) max(k-7,0) levels + the leaf block */
static size_t bit_arrays(const struct orc_prog *P, int k);
static void layout(const orc_prog *P, size_t count, layout_t *L)
{
    size_t off = 0;
    L->s16 = rup256(count * 16); L->s8 = rup256(count * 8);
    if (P->variant) {
        /* one tree per view width, in width order: k < n -> bit-DCF arrays (root, k levels, VCW bits);
         * k = n -> vector-DCF arrays with p = 1 (root, n levels of {sCW, VCW}, fin) */
        int pk = P->xpoly ? (int)P->S.d + 1 : 1;          /* payload words of the n-bit key: (1, -r, .., (-r)^d) with bit 2 */
        L->lvl_stride = L->s16 + (size_t)pk * L->s8;
        for (int w = 0; w < P->n_w; w++) {
            if (P->wk[w] < P->n) {
                L->bt_root[w] = off; off += L->s16;
                L->bt_cw[w] = off; off += L->s16 * bit_arrays(P, P->wk[w]);
                L->bt_vb[w] = off; off += L->s8;
            } else {
                L->vt_root[1] = off; off += L->s16;
                L->vt_lvl[1] = off; off += L->lvl_stride * (size_t)P->n;
                L->vt_fin[1] = off; off += (size_t)pk * L->s8;
            }
        }
    }
    for (int t = 0; t < P->T && !P->variant; t++) {
        L->bt_root[t] = off; off += L->s16;
        L->bt_cw[t] = off; off += L->s16 * bit_arrays(P, P->atoms[t].k);
        L->bt_vb[t] = off; off += L->s8;
    }
    if (!P->variant) L->lvl_stride = L->s16 + (size_t)P->p * L->s8;
    if (P->has_lut && !P->variant) {
        L->lut_c = off; off += (size_t)P->p * L->s8;
        for (int j = 1; j < P->M; j++) {
            L->vt_root[j] = off; off += L->s16;
            L->vt_lvl[j] = off; off += L->lvl_stride * (size_t)P->n;
            L->vt_fin[j] = off; off += (size_t)P->p * L->s8;
        }
    }
    L->rin = off; off += L->s8;
    L->rout = off; if (P->S.mask_output) off += (size_t)P->n_out_a * L->s8;
    L->ka = off; off += (size_t)P->S.n_kappa_a * L->s8;
    L->rpow = off; if (P->variant && P->xpoly) off += (size_t)P->S.d * L->s8;     /* [(-r)^t], t = 1..d (DESIGN 11) */
    L->kb = off; if (P->n_kb > 0) off += L->s8;
    L->beaver = off; off += (size_t)P->ma_word[P->MA] * L->s8;
    L->andt = off; if (P->MB > 0) off += 3 * L->s8;
    L->b2a_bits = off; if (P->GMIX > 0) off += L->s8;
    L->b2a_a = off; off += (size_t)P->GMIX * L->s8;
    L->a2b_rho = off; off += (size_t)P->GA2B * L->s8;                      /* A2B (DESIGN 15): [rho_i], one word of <bit_j(rho_i)>, */
    L->a2b_bits = off; if (P->GA2B > 0) off += L->s8;                      /* then one j_i-bit comparison key per node             */
    for (int i = 0; i < P->GA2B; i++) {
        L->a2b_root[i] = off; off += L->s16;
        L->a2b_cw[i] = off; off += L->s16 * bit_arrays(P, P->a2b_bit[i]);
        L->a2b_vb[i] = off; off += L->s8;
    }
    L->total = off;
}
static size_t bit_arrays(const orc_prog *P, int k) { return P->et ? (size_t)et_levels(k) + 1 : (size_t)k; }
size_t orc_key_bytes(const orc_prog *P, size_t count) { layout_t L; layout(P, count, &L); return L.total; }

/* ------------------------------------------------------------------------- */
/* 9. Deterministic randomness: R(e, slot) =                    */
/*    AES128_{seed || ~seed}(LE64(e) || LE64(slot)), e = GLOBAL element index. */
/* ------------------------------------------------------------------------- */
enum {
    SLOT_BT_ROOT = 0x1000, SLOT_VT_ROOT = 0x2000, SLOT_LUT_C = 0x3000, SLOT_RIN = 0x4000, SLOT_ROUT = 0x4100,
    SLOT_KA = 0x5000, SLOT_RPOW = 0x5400, SLOT_KB = 0x5800, SLOT_BV_AB = 0x6000, SLOT_BV_AB0 = 0x6800, SLOT_BV_C0 = 0x7000,
    SLOT_AND_AB = 0x8000, SLOT_AND_AB0 = 0x8001, SLOT_AND_C0 = 0x8002, SLOT_B2A = 0x9000, SLOT_B2A_A0 = 0x9100,
    SLOT_A2B_RHO = 0xB000, SLOT_A2B_RHO0 = 0xB100, SLOT_A2B_BITS = 0xB200, SLOT_A2B_ROOT = 0x1800
};
static void rnd(const aes_ks *ks, u64 e, u64 slot, u8 out[16])
{
    u8 in[16];
    put64(in, e); put64(in + 8, slot);
    aes_encrypt(ks, in, out);
}
static void seed_ks(u64 seed, aes_ks *ks)
{
    u8 key[16];
    put64(key, seed); put64(key + 8, ~seed);
    aes_expand(key, ks);
}

/* ------------------------------------------------------------------------- */
/* 10. keygen: dealer, per element (section 5.2)                     */
/* ------------------------------------------------------------------------- */
static void st16(u8 *base, size_t off, size_t e, const u8 *v) { memcpy(base + off + e * 16, v, 16); }
static void st8(u8 *base, size_t off, size_t e, u64 v) { put64(base + off + e * 8, v); }
static u64 ld8(const u8 *base, size_t off, size_t e) { return le64(base + off + e * 8); }

void orc_keygen(const orc_prog *P, const u64 *r_in, const u64 *r_out, u64 seed, u64 first_elem, size_t count,
                u8 *key0, u8 *key1)
{
    layout_t L; layout(P, count, &L);
    aes_ks ks; seed_ks(seed, &ks);
    const orc_spec *S = &P->S;
    u64 mask = P->mask;
    int n = P->n, p = P->p;
    u8 *key[2] = { key0, key1 };
    memset(key0, 0, L.total); memset(key1, 0, L.total);
    bitkey *bk0 = malloc(sizeof *bk0), *bk1 = malloc(sizeof *bk1);
    veckey *vk0 = malloc(sizeof *vk0), *vk1 = malloc(sizeof *vk1);
    for (size_t e = 0; e < count; e++) {
        u64 ge = first_elem + e;
        u64 r = r_in[e] & mask;
        u8 rb[16], rb1[16];
        /* ---- packed comparison instance: one bit-DCF per atom ---- */
        u64 kbits = 0;
        if (P->variant) {                                               /* DESIGN 9: one key per view width, threshold r_k */
            for (int w = 0; w < P->n_w; w++) {
                int k = P->wk[w];
                if (k < n) {
                    rnd(&ks, ge, SLOT_BT_ROOT + 2 * w, rb); rnd(&ks, ge, SLOT_BT_ROOT + 2 * w + 1, rb1);
                    if (P->et) dcf_bit_gen_et(k, r & low_mask(k), rb, rb1, bk0, bk1);
                    else dcf_bit_gen(k, r & low_mask(k), rb, rb1, bk0, bk1);
                    bitkey *bk[2] = { bk0, bk1 };
                    for (int b = 0; b < 2; b++) {
                        st16(key[b], L.bt_root[w], e, bk[b]->root);
                        for (int i = 0; i < (int)bit_arrays(P, k); i++) st16(key[b], L.bt_cw[w] + (size_t)i * L.s16, e, bk[b]->cw[i]);
                        st8(key[b], L.bt_vb[w], e, bk[b]->vbits);
                    }
                } else {
                    int pk = P->xpoly ? (int)S->d + 1 : 1;
                    u64 pw[PMAX]; pw[0] = 1 & mask;                      /* payload (1, -r, (-r)^2, ..) */
                    for (int t = 1; t < pk; t++) pw[t] = (pw[t - 1] * ((u64)0 - r)) & mask;
                    rnd(&ks, ge, SLOT_VT_ROOT + 2, rb); rnd(&ks, ge, SLOT_VT_ROOT + 3, rb1);
                    dcf_vec_gen(n, pk, mask, r, pw, rb, rb1, vk0, vk1);
                    veckey *vk[2] = { vk0, vk1 };
                    for (int b = 0; b < 2; b++) {
                        st16(key[b], L.vt_root[1], e, vk[b]->root);
                        for (int i = 0; i < n; i++) {
                            size_t lo = L.vt_lvl[1] + (size_t)i * L.lvl_stride;
                            st16(key[b], lo, e, vk[b]->scw[i]);
                            for (int t = 0; t < pk; t++) st8(key[b], lo + L.s16 + (size_t)t * L.s8, e, vk[b]->vcw[i][t]);
                        }
                        for (int t = 0; t < pk; t++) st8(key[b], L.vt_fin[1] + (size_t)t * L.s8, e, vk[b]->fin[t]);
                    }
                    for (int t = 1; t < pk; t++) {                      /* additive shares of (-r)^t */
                        rnd(&ks, ge, SLOT_RPOW + t, rb);
                        u64 s0 = le64(rb) & mask;
                        st8(key0, L.rpow + (size_t)(t - 1) * L.s8, e, s0); st8(key1, L.rpow + (size_t)(t - 1) * L.s8, e, (pw[t] - s0) & mask);
                    }
                }
            }
        }
        for (int t = 0; t < P->T && !P->variant; t++) {
            const atom_t *a = &P->atoms[t];
            u64 rk = r & low_mask(a->k);
            u64 theta = rk;
            if (a->is_theta) {
                u128 sum = (u128)rk + a->beta;                          /* Lemma 4.3: theta, carry w */
                theta = (u64)(sum & low_mask(a->k));
                int w = (sum >> a->k) ? 1 : 0;
                kbits |= (u64)w << a->carry_idx;
            }
            rnd(&ks, ge, SLOT_BT_ROOT + 2 * t, rb); rnd(&ks, ge, SLOT_BT_ROOT + 2 * t + 1, rb1);
            if (P->et) dcf_bit_gen_et(a->k, theta, rb, rb1, bk0, bk1);
            else dcf_bit_gen(a->k, theta, rb, rb1, bk0, bk1);
            bitkey *bk[2] = { bk0, bk1 };
            for (int b = 0; b < 2; b++) {
                st16(key[b], L.bt_root[t], e, bk[b]->root);
                for (int i = 0; i < (int)bit_arrays(P, a->k); i++) st16(key[b], L.bt_cw[t] + (size_t)i * L.s16, e, bk[b]->cw[i]);
                st8(key[b], L.bt_vb[t], e, bk[b]->vbits);
            }
        }
        for (u32 t = 0; t < S->n_kappa_b; t++) kbits |= (u64)kappa_b_value(S, (int)t, r) << (P->n_carry + t);
        /* ---- interval lookup instance (Protocol 3 (1),(5); reading S2: sum of M-1 vector DCFs) ---- */
        if (P->has_lut && !P->variant) {
            u128 B[MMAX + 2]; int ord[MMAX + 1], M;
            protocol3(n, P->m, S->alpha, r, B, ord, &M);
            u64 v[MMAX + 1][PMAX];
            for (int j = 0; j < M; j++) {                               /* payloads v_j (lines 31-33) */
                int w = 0;
                for (u32 q = 0; q < S->r * (S->d + 1); q++)
                    v[j][w++] = P->xpoly ? shifted_coeff(S, ord[j], (int)(q / (S->d + 1)), (int)(S->d - q % (S->d + 1)), r, mask)
                                         : S->coeff[(size_t)ord[j] * S->r * (S->d + 1) + q] & mask;
                for (u32 q = 0; q < S->p_aux; q++) v[j][w++] = S->aux[(size_t)ord[j] * S->p_aux + q] & mask;
            }
            for (int w = 0; w < p; w++) {                               /* constant term v_{M-1}, additively split */
                rnd(&ks, ge, SLOT_LUT_C + w, rb);
                u64 c0 = le64(rb) & mask, c1 = (v[M - 1][w] - c0) & mask;
                st8(key0, L.lut_c + (size_t)w * L.s8, e, c0);
                st8(key1, L.lut_c + (size_t)w * L.s8, e, c1);
            }
            for (int j = 1; j < M; j++) {
                u64 delta[PMAX];
                for (int w = 0; w < p; w++) delta[w] = (v[j - 1][w] - v[j][w]) & mask;
                rnd(&ks, ge, SLOT_VT_ROOT + 2 * j, rb); rnd(&ks, ge, SLOT_VT_ROOT + 2 * j + 1, rb1);
                dcf_vec_gen(n, p, mask, (u64)B[j], delta, rb, rb1, vk0, vk1);
                veckey *vk[2] = { vk0, vk1 };
                for (int b = 0; b < 2; b++) {
                    st16(key[b], L.vt_root[j], e, vk[b]->root);
                    for (int i = 0; i < n; i++) {
                        size_t lo = L.vt_lvl[j] + (size_t)i * L.lvl_stride;
                        st16(key[b], lo, e, vk[b]->scw[i]);
                        for (int w = 0; w < p; w++) st8(key[b], lo + L.s16 + (size_t)w * L.s8, e, vk[b]->vcw[i][w]);
                    }
                    for (int w = 0; w < p; w++) st8(key[b], L.vt_fin[j] + (size_t)w * L.s8, e, vk[b]->fin[w]);
                }
            }
        }
        /* ---- masks, instance constants, correlated randomness ---- */
        rnd(&ks, ge, SLOT_RIN, rb);
        { u64 s0 = le64(rb) & mask; st8(key0, L.rin, e, s0); st8(key1, L.rin, e, (r - s0) & mask); }
        if (S->mask_output) for (int j = 0; j < P->n_out_a; j++) {
            rnd(&ks, ge, SLOT_ROUT + j, rb);
            u64 ro = r_out[(size_t)j * count + e] & mask, s0 = le64(rb) & mask;
            st8(key0, L.rout + (size_t)j * L.s8, e, s0); st8(key1, L.rout + (size_t)j * L.s8, e, (ro - s0) & mask);
        }
        for (u32 t = 0; t < S->n_kappa_a; t++) {
            rnd(&ks, ge, SLOT_KA + t, rb);
            u64 val = kappa_a_value(S, (int)t, r) & mask, s0 = le64(rb) & mask;
            st8(key0, L.ka + (size_t)t * L.s8, e, s0); st8(key1, L.ka + (size_t)t * L.s8, e, (val - s0) & mask);
        }
        if (P->n_kb > 0) {
            rnd(&ks, ge, SLOT_KB, rb);
            u64 s0 = le64(rb) & low_mask(P->n_kb);
            st8(key0, L.kb, e, s0); st8(key1, L.kb, e, kbits ^ s0);
        }
        for (int i = 0; i < P->MA; i++) {                               /* Beaver triples (a, b, c = ab) */
            rnd(&ks, ge, SLOT_BV_AB + i, rb);
            u64 a = le64(rb) & mask, b = le64(rb + 8) & mask, c = (a * b) & mask;
            rnd(&ks, ge, SLOT_BV_AB0 + i, rb);
            u64 a0 = le64(rb) & mask, b0 = le64(rb + 8) & mask;
            rnd(&ks, ge, SLOT_BV_C0 + i, rb);
            u64 c0 = le64(rb) & mask;
            size_t o = L.beaver + (size_t)P->ma_word[i] * L.s8;
            if (P->ma_is_x[i]) {                                        /* (b, c = b r_in): DESIGN 10 */
                u64 cx = (b * r) & mask;
                st8(key0, o, e, b0); st8(key0, o + L.s8, e, c0);
                st8(key1, o, e, (b - b0) & mask); st8(key1, o + L.s8, e, (cx - c0) & mask);
                continue;
            }
            st8(key0, o, e, a0); st8(key0, o + L.s8, e, b0); st8(key0, o + 2 * L.s8, e, c0);
            st8(key1, o, e, (a - a0) & mask); st8(key1, o + L.s8, e, (b - b0) & mask); st8(key1, o + 2 * L.s8, e, (c - c0) & mask);
        }
        if (P->MB > 0) {                                                /* AND triples, bit idx of three words */
            u64 bm = low_mask(P->MB);
            rnd(&ks, ge, SLOT_AND_AB, rb);
            u64 a = le64(rb) & bm, b = le64(rb + 8) & bm, c = a & b;
            rnd(&ks, ge, SLOT_AND_AB0, rb);
            u64 a0 = le64(rb) & bm, b0 = le64(rb + 8) & bm;
            rnd(&ks, ge, SLOT_AND_C0, rb);
            u64 c0 = le64(rb) & bm;
            st8(key0, L.andt, e, a0); st8(key0, L.andt + L.s8, e, b0); st8(key0, L.andt + 2 * L.s8, e, c0);
            st8(key1, L.andt, e, a ^ a0); st8(key1, L.andt + L.s8, e, b ^ b0); st8(key1, L.andt + 2 * L.s8, e, c ^ c0);
        }
        if (P->GMIX > 0) {                                              /* B2A pairs (<rho>, [rho]) */
            u64 bm = low_mask(P->GMIX);
            rnd(&ks, ge, SLOT_B2A, rb);
            u64 rho = le64(rb) & bm, rho0 = le64(rb + 8) & bm;
            st8(key0, L.b2a_bits, e, rho0); st8(key1, L.b2a_bits, e, rho ^ rho0);
            for (int i = 0; i < P->GMIX; i++) {
                rnd(&ks, ge, SLOT_B2A_A0 + i, rb);
                u64 s0 = le64(rb) & mask, val = (rho >> i) & 1;
                st8(key0, L.b2a_a + (size_t)i * L.s8, e, s0); st8(key1, L.b2a_a + (size_t)i * L.s8, e, (val - s0) & mask);
            }
        }
        if (P->GA2B > 0) {                                              /* A2B material (DESIGN 15): mask rho, <bit_j(rho)>, f_{rho mod 2^j, 1} */
            u64 rbits = 0;
            for (int i = 0; i < P->GA2B; i++) {
                int j = P->a2b_bit[i];
                rnd(&ks, ge, SLOT_A2B_RHO + i, rb);
                u64 rho = le64(rb) & mask;
                rnd(&ks, ge, SLOT_A2B_RHO0 + i, rb);
                u64 s0 = le64(rb) & mask;
                st8(key0, L.a2b_rho + (size_t)i * L.s8, e, s0); st8(key1, L.a2b_rho + (size_t)i * L.s8, e, (rho - s0) & mask);
                rbits |= ((rho >> j) & 1) << i;
                rnd(&ks, ge, SLOT_A2B_ROOT + 2 * i, rb); rnd(&ks, ge, SLOT_A2B_ROOT + 2 * i + 1, rb1);
                if (P->et) dcf_bit_gen_et(j, rho & low_mask(j), rb, rb1, bk0, bk1);
                else dcf_bit_gen(j, rho & low_mask(j), rb, rb1, bk0, bk1);
                bitkey *bk[2] = { bk0, bk1 };
                for (int b = 0; b < 2; b++) {
                    st16(key[b], L.a2b_root[i], e, bk[b]->root);
                    for (int l = 0; l < (int)bit_arrays(P, j); l++) st16(key[b], L.a2b_cw[i] + (size_t)l * L.s16, e, bk[b]->cw[l]);
                    st8(key[b], L.a2b_vb[i], e, bk[b]->vbits);
                }
            }
            rnd(&ks, ge, SLOT_A2B_BITS, rb);
            u64 b0 = le64(rb) & low_mask(P->GA2B);
            st8(key0, L.a2b_bits, e, b0); st8(key1, L.a2b_bits, e, rbits ^ b0);
        }
    }
    free(bk0); free(bk1); free(vk0); free(vk1);
}

/* ------------------------------------------------------------------------- */
/* 11. eval_cmp / eval_lut: local, per party               */
/* ------------------------------------------------------------------------- */
static void ld16(const u8 *base, size_t off, size_t e, u8 *v) { memcpy(v, base + off + e * 16, 16); }

/* variant 1: A[w][j] = Eval_b(key_w, (xhat + delta_j) mod 2^k), every point from the root (plain definition) */
static void sp_eval_points(int party, const orc_prog *P, const u8 *key, const layout_t *L, size_t e, u64 xh,
                           bitkey *bk, veckey *vk, u64 A[8][2 * TMAX + 2], u64 AV[2 * TMAX + 2][PMAX])
{
    int n = P->n;
    int pk = P->xpoly ? (int)P->S.d + 1 : 1;
    for (int w = 0; w < P->n_w; w++) {
        int k = P->wk[w];
        u64 km = low_mask(k);
        if (k < n) {
            ld16(key, L->bt_root[w], e, bk->root);
            for (int i = 0; i < (int)bit_arrays(P, k); i++) ld16(key, L->bt_cw[w] + (size_t)i * L->s16, e, bk->cw[i]);
            bk->vbits = ld8(key, L->bt_vb[w], e);
            for (int j = 0; j < P->w_npts[w]; j++)
                A[w][j] = (u64)(P->et ? dcf_bit_eval_et(party, k, bk, (xh + P->w_delta[w][j]) & km) : dcf_bit_eval(party, k, bk, (xh + P->w_delta[w][j]) & km));
        } else {
            ld16(key, L->vt_root[1], e, vk->root);
            for (int i = 0; i < n; i++) {
                size_t lo = L->vt_lvl[1] + (size_t)i * L->lvl_stride;
                ld16(key, lo, e, vk->scw[i]);
                for (int t = 0; t < pk; t++) vk->vcw[i][t] = ld8(key, lo + L->s16 + (size_t)t * L->s8, e);
            }
            for (int t = 0; t < pk; t++) vk->fin[t] = ld8(key, L->vt_fin[1] + (size_t)t * L->s8, e);
            for (int j = 0; j < P->w_npts[w]; j++) {
                dcf_vec_eval(party, n, pk, P->mask, vk, (xh + P->w_delta[w][j]) & km, AV[j]);
                A[w][j] = AV[j][0];                                     /* component 0 = share of I[u_j < r] */
            }
        }
    }
}
/* share of the predicate atom t: e - b + a in R (k = n) or e ^ b ^ a (k < n); r-atom: b itself */
static u64 sp_atom_share(int party, const orc_prog *P, int t, u64 xh, u64 A[8][2 * TMAX + 2])
{
    const atom_t *a = &P->atoms[t];
    int w = P->atom_w[t];
    u64 km = low_mask(a->k);
    u64 b = A[w][P->atom_ib[t]];
    if (!a->is_theta) return b;
    u64 h = (xh + a->c) & km;
    u64 pub = (party == 0 && h < a->beta) ? 1 : 0;
    u64 av = A[w][P->atom_ia[t]];
    return a->k < P->n ? (pub ^ b ^ av) : ((pub - b + av) & P->mask);
}
static void sp_eval(int party, const orc_prog *P, const u8 *key, const u64 *xhat, size_t count, u64 *bits_out, u64 *coeff_out)
{
    layout_t L; layout(P, count, &L);
    bitkey *bk = malloc(sizeof *bk); veckey *vk = malloc(sizeof *vk);
    u64 (*A)[2 * TMAX + 2] = malloc(sizeof(u64) * 8 * (2 * TMAX + 2));
    u64 (*AV)[PMAX] = malloc(sizeof(u64) * PMAX * (2 * TMAX + 2));
    const orc_spec *S = &P->S;
    u32 nc = S->r * (S->d + 1);
    for (size_t e = 0; e < count; e++) {
        u64 xh = xhat[e] & P->mask;
        sp_eval_points(party, P, key, &L, e, xh, bk, vk, A, AV);
        if (bits_out) {
            u64 word = 0;
            for (int t = 0; t < P->T; t++) word |= (sp_atom_share(party, P, t, xh, A) & 1) << t;   /* LSB of an additive share of a bit = XOR share */
            bits_out[e] = word;
        }
        if (coeff_out && P->has_lut) {
            /* v_{i*} = v_{m-1} + sum_{i=1}^{m-1} (v_{i-1} - v_i) I[x < alpha_i]  (Lemma D.1 telescoped); v_i public */
            for (int wd = 0; wd < P->p && P->xpoly; wd++) {
                /* DESIGN 11: coefficient of xhat^j of P_{i*}(xhat - r):  c'_j = sum_t sum_i J_i (-r)^t c_{i,j+t} C(j+t, j), with
                 * [I[x<alpha_i] (-r)^t] = e_i [(-r)^t] - B[t] + A_i[t]  (B, A_i = the vector key at the offsets 0, -alpha_i) */
                int d = (int)S->d, q = wd / (d + 1), j = d - wd % (d + 1), is_aux = wd >= (int)nc;
                u64 acc = 0;
                for (int t = 0; t <= (is_aux ? 0 : d - j); t++) {
                    u64 rp = t == 0 ? (party == 0 ? 1 : 0) : ld8(key, L.rpow + (size_t)(t - 1) * L.s8, e);
                    u64 wprev = 0;
                    for (int i = 0; i < P->m; i++) {
                        u64 wi = is_aux ? S->aux[(size_t)i * S->p_aux + (wd - nc)]
                                        : S->coeff[((size_t)i * S->r + q) * (d + 1) + (d - (j + t))] * binom(j + t, j);
                        wi &= P->mask;
                        if (i) {
                            int ta = P->alpha_atom[i];
                            u64 ei = (xh < S->alpha[i - 1]) ? 1 : 0;
                            u64 sh = ei * rp - AV[P->atom_ib[ta]][t] + AV[P->atom_ia[ta]][t];
                            acc += (wprev - wi) * sh;
                        }
                        if (i == P->m - 1) acc += wi * rp;
                        wprev = wi;
                    }
                }
                coeff_out[(size_t)wd * count + e] = acc & P->mask;
            }
            if (P->dense) {
                /* Dense-table lookup (DESIGN 14): T[u] = payload of the interval that contains u, u = 0..N-1 -- the operator as a
                 * table of 2^n entries.  With A_b(v) = Eval_b(key, v) the share of I[v < r] at EVERY point v of the domain and
                 * D[a] = T[a-1] - T[a]:   T[x] = T[xhat] - I[xhat < r] (T[0] - T[N-1]) + sum_{a=1}^{N-1} D[a] I[(xhat - a) mod N < r]
                 * (the variant-1 identity with every point of the ring as a boundary).  Work and shape depend on n only. */
                u64 N = (u64)1 << P->n;
                u64 acc[PMAX] = { 0 };
                for (u64 v = 0; v < N; v++) {
                    u64 Av[PMAX];
                    dcf_vec_eval(party, P->n, 1, P->mask, vk, v, Av);
                    u64 a = (xh - v) & P->mask;                        /* v = xhat - a */
                    for (int wd = 0; wd < P->p; wd++) {
                        u64 T0 = (wd < (int)nc ? S->coeff[wd] : S->aux[wd - nc]) & P->mask;
                        int il = P->m - 1;
                        u64 TN = (wd < (int)nc ? S->coeff[(size_t)il * nc + wd] : S->aux[(size_t)il * S->p_aux + (wd - nc)]) & P->mask;
                        if (a == 0) { acc[wd] -= Av[0] * (T0 - TN); continue; }          /* the term B = A(xhat) */
                        int ia = plain_interval(S, a), ib = plain_interval(S, a - 1);
                        u64 Ta = (wd < (int)nc ? S->coeff[(size_t)ia * nc + wd] : S->aux[(size_t)ia * S->p_aux + (wd - nc)]) & P->mask;
                        u64 Tb = (wd < (int)nc ? S->coeff[(size_t)ib * nc + wd] : S->aux[(size_t)ib * S->p_aux + (wd - nc)]) & P->mask;
                        acc[wd] += (Tb - Ta) * Av[0];
                    }
                }
                int ix = plain_interval(S, xh);
                for (int wd = 0; wd < P->p; wd++) {
                    u64 Tx = (wd < (int)nc ? S->coeff[(size_t)ix * nc + wd] : S->aux[(size_t)ix * S->p_aux + (wd - nc)]) & P->mask;
                    coeff_out[(size_t)wd * count + e] = (acc[wd] + (party == 0 ? Tx : 0)) & P->mask;
                }
                continue;
            }
            for (int wd = 0; wd < P->p && !P->xpoly; wd++) {
                u64 acc = 0;
                for (int i = 0; i < P->m; i++) {
                    u64 vi = (wd < (int)nc ? S->coeff[(size_t)i * nc + wd] : S->aux[(size_t)i * S->p_aux + (wd - nc)]) & P->mask;
                    u64 vprev = i ? ((wd < (int)nc ? S->coeff[(size_t)(i - 1) * nc + wd] : S->aux[(size_t)(i - 1) * S->p_aux + (wd - nc)]) & P->mask) : 0;
                    if (i) acc += (vprev - vi) * sp_atom_share(party, P, P->alpha_atom[i], xh, A);
                    if (i == P->m - 1 && party == 0) acc += vi;
                }
                coeff_out[(size_t)wd * count + e] = acc & P->mask;
            }
        }
    }
    free(bk); free(vk); free(A); free(AV);
}

void orc_eval_cmp(int party, const orc_prog *P, const u8 *key, const u64 *xhat, size_t count, u64 *bits_out)
{
    if (P->variant) { if (P->T) sp_eval(party, P, key, xhat, count, bits_out, NULL); return; }
    layout_t L; layout(P, count, &L);
    bitkey *bk = malloc(sizeof *bk);
    for (size_t e = 0; e < count; e++) {
        u64 word = 0;
        for (int t = 0; t < P->T; t++) {
            const atom_t *a = &P->atoms[t];
            ld16(key, L.bt_root[t], e, bk->root);
            for (int i = 0; i < (int)bit_arrays(P, a->k); i++) ld16(key, L.bt_cw[t] + (size_t)i * L.s16, e, bk->cw[i]);
            bk->vbits = ld8(key, L.bt_vb[t], e);
            /* view_{k,c}(xhat) = ((xhat mod 2^k) + c) mod 2^k */
            u64 u = ((xhat[e] & low_mask(a->k)) + a->c) & low_mask(a->k);
            word |= (u64)(P->et ? dcf_bit_eval_et(party, a->k, bk, u) : dcf_bit_eval(party, a->k, bk, u)) << t;
        }
        bits_out[e] = word;
    }
    free(bk);
}

void orc_eval_lut(int party, const orc_prog *P, const u8 *key, const u64 *xhat, size_t count, u64 *coeff_out)
{
    if (P->variant) { sp_eval(party, P, key, xhat, count, NULL, coeff_out); return; }
    layout_t L; layout(P, count, &L);
    if (!P->has_lut) return;
    veckey *vk = malloc(sizeof *vk);
    int n = P->n, p = P->p;
    for (size_t e = 0; e < count; e++) {
        u64 acc[PMAX];
        for (int w = 0; w < p; w++) acc[w] = ld8(key, L.lut_c + (size_t)w * L.s8, e);
        for (int j = 1; j < P->M; j++) {
            ld16(key, L.vt_root[j], e, vk->root);
            for (int i = 0; i < n; i++) {
                size_t lo = L.vt_lvl[j] + (size_t)i * L.lvl_stride;
                ld16(key, lo, e, vk->scw[i]);
                for (int w = 0; w < p; w++) vk->vcw[i][w] = ld8(key, lo + L.s16 + (size_t)w * L.s8, e);
            }
            for (int w = 0; w < p; w++) vk->fin[w] = ld8(key, L.vt_fin[j] + (size_t)w * L.s8, e);
            u64 out[PMAX];
            dcf_vec_eval(party, n, p, P->mask, vk, xhat[e] & P->mask, out);
            for (int w = 0; w < p; w++) acc[w] = (acc[w] + out[w]) & P->mask;
        }
        for (int w = 0; w < p; w++) coeff_out[(size_t)w * count + e] = acc[w];
    }
    free(vk);
}

/* ------------------------------------------------------------------------- */
/* 12. post-processing (subprotocols: reading S6)           */
/*     Message buffer of one party: for round q = 0..rounds-1, for each Beaver */
/*     mult of that round in program order the arrays E[count], F[count], then */
/*     (if the round opens bits) one array of packed bits; arrays padded to    */
/*     256 B.  Stateless: a call for round q replays rounds < q from msg_in.   */
/* ------------------------------------------------------------------------- */
size_t orc_post_msg_bytes(const orc_prog *P, size_t count, int round)
{
    size_t s8 = rup256(count * 8);
    if (round < 0 || round >= P->rounds) return 0;
    return s8 * ((size_t)P->r_narr[round] + (P->r_nbits[round] ? 1 : 0));
}
int orc_post_rounds(const orc_prog *P) { return P->rounds; }
/* algorithmic online bits per element per party: n (xhat, Protocol 1) + 2n per Beaver + 2 per AND + 1 per B2A
 * (+ n per masked output) */
size_t orc_online_bits(const orc_prog *P)
{
    size_t arrs = 0;
    for (int q = 0; q < P->rounds; q++) arrs += (size_t)P->r_narr[q];
    return (size_t)P->n + (size_t)P->n * arrs + (size_t)2 * P->MB + (size_t)P->GMIX
         + (P->S.mask_output ? (size_t)P->n * P->n_out_a : 0);
}

void orc_post(int party, const orc_prog *P, const u8 *key, const u64 *xhat, const u64 *bits, const u64 *coeff,
              size_t count, int round, const u8 *msg_in, u8 *msg_out, u64 *y_out, u64 *z_out)
{
    layout_t L; layout(P, count, &L);
    u64 mask = P->mask;
    size_t s8 = rup256(count * 8);
    size_t roff[17]; roff[0] = 0;
    for (int q = 0; q < P->rounds; q++) roff[q + 1] = roff[q] + orc_post_msg_bytes(P, count, q);
    u64 *A = malloc(sizeof(u64) * REGMAX); u8 *Bv = malloc(REGMAX);
    for (size_t e = 0; e < count; e++) {
        u64 xh = xhat[e] & mask;
        int mulpos[16] = { 0 }, bitpos[16] = { 0 };
        u64 outbits[16] = { 0 };
        u64 zword = 0;
        for (int i = 0; i < P->nops; i++) {
            const cop_t *o = &P->ops[i];
            switch (o->op) {
            case C_B_CONST: Bv[o->dst] = party == 0 ? (u8)(o->imm & 1) : 0; break;
            case C_B_ATOM: Bv[o->dst] = (u8)((bits[e] >> o->a) & 1); break;
            case C_B_KAPPA: Bv[o->dst] = (u8)((ld8(key, L.kb, e) >> o->a) & 1); break;
            case C_B_XHAT: Bv[o->dst] = party == 0 ? (u8)((xh >> o->a) & 1) : 0; break;
            case C_B_NOT: Bv[o->dst] = Bv[o->a] ^ (party == 0 ? 1 : 0); break;
            case C_B_XOR: Bv[o->dst] = Bv[o->a] ^ Bv[o->b]; break;
            case C_B_ANDPUB: Bv[o->dst] = Bv[o->a] & (u8)(((xh >> o->b) & 1) ^ (o->imm & 1)); break;
            case C_B_OUT: zword |= (u64)Bv[o->a] << o->dst; break;
            case C_B_AND: {  /* open d = u^a, e = v^b; z_b = [b=0](d&e) ^ (d&b_b) ^ (e&a_b) ^ c_b */
                int q = o->round, pos = bitpos[q]; bitpos[q] += 2;
                u8 ta = (u8)((ld8(key, L.andt, e) >> o->idx) & 1), tb = (u8)((ld8(key, L.andt + L.s8, e) >> o->idx) & 1),
                   tc = (u8)((ld8(key, L.andt + 2 * L.s8, e) >> o->idx) & 1);
                u8 dm = Bv[o->a] ^ ta, em = Bv[o->b] ^ tb;
                if (q == round) outbits[q] |= ((u64)dm << pos) | ((u64)em << (pos + 1));
                if (q < round) {
                    u64 other = ld8(msg_in, roff[q] + (size_t)P->r_narr[q] * s8, e);
                    u8 dd = dm ^ (u8)((other >> pos) & 1), ee = em ^ (u8)((other >> (pos + 1)) & 1);
                    Bv[o->dst] = (u8)((party == 0 ? (dd & ee) : 0) ^ (dd & tb) ^ (ee & ta) ^ tc);
                } else Bv[o->dst] = 0;
                break; }
            case C_A_CONST: A[o->dst] = party == 0 ? (o->imm & mask) : 0; break;
            case C_A_X:  /* Protocol 2: x_0 = xhat - r_0, x_1 = -r_1 */
                A[o->dst] = party == 0 ? (xh - ld8(key, L.rin, e)) & mask : ((u64)0 - ld8(key, L.rin, e)) & mask; break;
            case C_A_COEFF: A[o->dst] = coeff[(size_t)o->a * count + e] & mask; break;
            case C_A_KAPPA: A[o->dst] = ld8(key, L.ka + (size_t)o->a * L.s8, e); break;
            case C_A_XHAT_SHR: A[o->dst] = party == 0 ? (o->a >= 64 ? 0 : xh >> o->a) : 0; break;
            case C_A_ADD: A[o->dst] = (A[o->a] + A[o->b]) & mask; break;
            case C_A_SUB: A[o->dst] = (A[o->a] - A[o->b]) & mask; break;
            case C_A_MULC: A[o->dst] = (A[o->a] * o->imm) & mask; break;
            case C_A_MULXH: A[o->dst] = (A[o->a] * xh) & mask; break;
            case C_A_OUT: {
                u64 v = A[o->a];
                if (P->S.mask_output) v = (v + ld8(key, L.rout + (size_t)o->dst * L.s8, e)) & mask;   /* yhat share */
                if (round == P->rounds) y_out[(size_t)o->dst * count + e] = v;
                break; }
            case C_A_MUL: {  /* Beaver: open e = x-a, f = y-b; [xy]_b = [b=0]ef + e[b]_b + f[a]_b + [c]_b */
                int q = o->round, pos = mulpos[q]; mulpos[q] += 2;      /* pos = first array of this gate in round q */
                size_t to = L.beaver + (size_t)P->ma_word[o->idx] * L.s8;
                u64 ta = ld8(key, to, e), tb = ld8(key, to + L.s8, e), tc = ld8(key, to + 2 * L.s8, e);
                u64 em = (A[o->a] - ta) & mask, fm = (A[o->b] - tb) & mask;
                if (q == round) { st8(msg_out, roff[q] + (size_t)pos * s8, e, em); st8(msg_out, roff[q] + (size_t)(pos + 1) * s8, e, fm); }
                if (q < round) {
                    u64 E = (em + ld8(msg_in, roff[q] + (size_t)pos * s8, e)) & mask;
                    u64 F = (fm + ld8(msg_in, roff[q] + (size_t)(pos + 1) * s8, e)) & mask;
                    A[o->dst] = ((party == 0 ? E * F : 0) + E * tb + F * ta + tc) & mask;
                } else A[o->dst] = 0;
                break; }
            case C_A_MULX: { /* y * x with x = xhat - r_in, xhat public (DESIGN 10): material (b, c = b r_in); open f = y - b;
                              * [y x]_b = xhat [y]_b - f [r_in]_b - [c]_b */
                int q = o->round, pos = mulpos[q]; mulpos[q] += 1;
                size_t to = L.beaver + (size_t)P->ma_word[o->idx] * L.s8;
                u64 tb = ld8(key, to, e), tc = ld8(key, to + L.s8, e);
                u64 fm = (A[o->a] - tb) & mask;
                if (q == round) st8(msg_out, roff[q] + (size_t)pos * s8, e, fm);
                if (q < round) {
                    u64 F = (fm + ld8(msg_in, roff[q] + (size_t)pos * s8, e)) & mask;
                    A[o->dst] = (xh * A[o->a] - F * ld8(key, L.rin, e) - tc) & mask;
                } else A[o->dst] = 0;
                break; }
            case C_B_LSB: Bv[o->dst] = (u8)(A[o->a] & 1); break;             /* (e_0 + e_1) mod 2 = e_0 ^ e_1 on the low bit */
            case C_B_A2B: {  /* bit j of e (DESIGN 15): open ehat = e + rho; bit_j(e) = bit_j(ehat) ^ bit_j(rho) ^ I[ehat mod 2^j < rho mod 2^j] */
                int q = o->round, pos = mulpos[q]; mulpos[q] += 1;
                int j = (int)o->imm;
                u64 em = (A[o->a] + ld8(key, L.a2b_rho + (size_t)o->idx * L.s8, e)) & mask;
                if (q == round) st8(msg_out, roff[q] + (size_t)pos * s8, e, em);
                if (q < round) {
                    u64 E = (em + ld8(msg_in, roff[q] + (size_t)pos * s8, e)) & mask;
                    bitkey *bk = malloc(sizeof *bk);
                    ld16(key, L.a2b_root[o->idx], e, bk->root);
                    for (int l = 0; l < (int)bit_arrays(P, j); l++) ld16(key, L.a2b_cw[o->idx] + (size_t)l * L.s16, e, bk->cw[l]);
                    bk->vbits = ld8(key, L.a2b_vb[o->idx], e);
                    int c = P->et ? dcf_bit_eval_et(party, j, bk, E & low_mask(j)) : dcf_bit_eval(party, j, bk, E & low_mask(j));
                    free(bk);
                    u8 rb_ = (u8)((ld8(key, L.a2b_bits, e) >> o->idx) & 1);
                    Bv[o->dst] = (u8)((party == 0 ? (int)((E >> j) & 1) : 0) ^ rb_ ^ c);
                } else Bv[o->dst] = 0;
                break; }
            case C_A_B2A: {  /* open mu = z ^ rho; [z]_b = [b=0]mu + [rho]_b - 2 mu [rho]_b */
                int q = o->round, pos = bitpos[q]; bitpos[q] += 1;
                u8 rb = (u8)((ld8(key, L.b2a_bits, e) >> o->idx) & 1);
                u64 ra = ld8(key, L.b2a_a + (size_t)o->idx * L.s8, e);
                u8 mm = Bv[o->a] ^ rb;
                if (q == round) outbits[q] |= (u64)mm << pos;
                if (q < round) {
                    u64 other = ld8(msg_in, roff[q] + (size_t)P->r_narr[q] * s8, e);
                    u64 mu = (u64)(mm ^ (u8)((other >> pos) & 1));
                    A[o->dst] = ((party == 0 ? mu : 0) + ra - 2 * mu * ra) & mask;
                } else A[o->dst] = 0;
                break; }
            }
        }
        if (round < P->rounds && P->r_nbits[round])
            st8(msg_out, roff[round] + (size_t)P->r_narr[round] * s8, e, outbits[round]);
        if (round == P->rounds && P->n_out_b > 0) z_out[e] = zword;
    }
    free(A); free(Bv);
}

/* ------------------------------------------------------------------------- */
/* 13. Dealer randomness for the vector-block glue (oracle/blocks.py):         */
/*     lo/hi words of R(e, slot), e = first .. first+count-1 (DESIGN 4.5)      */
/* ------------------------------------------------------------------------- */
void orc_dealer_rand(u64 seed, u64 first, size_t count, u64 slot, u64 *lo, u64 *hi)
{
    aes_ks ks; seed_ks(seed, &ks);
    for (size_t i = 0; i < count; i++) {
        u8 rb[16];
        rnd(&ks, first + i, slot, rb);
        lo[i] = le64(rb); hi[i] = le64(rb + 8);
    }
}
/* [r_in] share of element e in a key buffer (for Protocol 1 in the block composition) */
void orc_rin_shares(const orc_prog *P, const u8 *key, size_t count, u64 *out)
{
    layout_t L; layout(P, count, &L);
    for (size_t e = 0; e < count; e++) out[e] = ld8(key, L.rin, e);
}
