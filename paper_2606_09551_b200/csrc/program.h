// program.h -- compiled gate type shared by the host compiler (compile.cpp) and the kernel launchers.
// Product code: independent of oracle/ (DESIGN.md section 3).  Format definitions: DESIGN.md section 4.
#pragma once
#include <cstddef>
#include <cstdint>
#include <map>
#include <mutex>
#include <vector>

#include "../../include/fusefss.h"

namespace fsk {

constexpr int kMaxAtoms = 64;      // T <= 64: one packed word of share bits per element
constexpr int kMaxP = 8;           // payload words p
constexpr int kMaxIntervals = 64;  // m < 64
constexpr int kMaxRounds = 16;
constexpr int kMaxAReg = 48;       // arithmetic registers after allocation (device local array)
constexpr int kMaxBReg = 128;      // bit registers after allocation (two 64-bit words per party)
constexpr int kMaxA2B = 8;         // interactive A2B nodes per gate

// One query of the packed comparison instance (Def I.1).
struct Atom {
    int k;              // view width k_t
    uint64_t c;         // view offset c_t
    int is_theta;       // 0: r-atom (threshold r mod 2^k), 1: theta-atom (threshold (r_k + beta) mod 2^k)
    uint64_t beta;
    int carry;          // index of the carry bit w_t inside kappa^B, -1 for r-atoms
};

// Post-processing instruction (DESIGN 4.3 "post program").  Interactive gates carry their gate number
// (`gate`), their round and their position inside that round's message (`pos`).
enum : uint8_t {
    I_B_CONST = 1, I_B_ATOM, I_B_KAPPA, I_B_XHAT, I_B_NOT, I_B_XOR, I_B_AND, I_B_ANDPUB, I_B_OUT,
    I_A_CONST, I_A_X, I_A_COEFF, I_A_KAPPA, I_A_XHAT_SHR, I_A_ADD, I_A_SUB, I_A_MULC, I_A_MUL, I_A_MULX, I_A_MULXH, I_A_B2A, I_A_OUT,
    I_B_LSB,            // B[dst] = bit 0 of the shared ring element A[a]: local (DESIGN 15)
    I_B_A2B             // B[dst] = bit imm >= 1 of A[a]: open A[a] + rho, then one imm-bit comparison key (DESIGN 15); gate = A2B index
};
struct Ins {
    uint8_t op;
    uint8_t round;      // interactive gates only
    uint16_t dst, a, b;
    uint16_t gate;      // Beaver / AND / B2A gate number
    uint16_t pos;       // Beaver: pair index inside the round; AND/B2A: first bit position inside the round's bit word
    uint32_t pad;
    uint64_t imm;       // constants; for I_A_MUL / I_A_MULX: first word of the gate's material inside the Beaver section
};
static_assert(sizeof(Ins) == 24, "Ins is uploaded to the device as-is");

// Byte offsets inside one party's key buffer (DESIGN 4.4).
struct Layout {
    size_t s16, s8;
    size_t bt_root[kMaxAtoms], bt_cw[kMaxAtoms], bt_vb[kMaxAtoms];
    size_t lut_c, vt_first, vt_stride, lvl_stride, vt_lvl_rel, vt_fin_rel;   // vector tree j at vt_first + (j-1)*vt_stride
    size_t rin, rout, ka, rpow, kb, beaver, andt, b2a_bits, b2a_a, total;
    size_t a2b_rho, a2b_bits, a2b_root[kMaxA2B], a2b_cw[kMaxA2B], a2b_vb[kMaxA2B];   // A2B material (DESIGN 15), after the B2A section
};

// variant 1: single-key shared-prefix construction
constexpr int kMaxWidths = 8;
constexpr int kMaxPoints = 2 * kMaxAtoms + 2;
struct SpPoint { uint64_t delta; uint64_t bitmask; };      // offset added to xhat; atoms whose bit flips with LSB(A_j)
struct SpCluster { int first, count, tail_bits, pad; };    // points [first, first+count) share their top n - tail_bits bits (two candidate prefixes)
struct SpWidth { int k, first_point, n_points, is_vec; };
struct SpProgram {
    int n_w = 0;
    SpWidth width[kMaxWidths];
    std::vector<SpPoint> points;        // all widths, width-major, sorted by signed delta inside a width
    int pk = 1;                         // payload words of the n-bit key: 1, or d+1 = (1, -r, .., (-r)^d) with variant bit 2
    std::vector<uint64_t> weights;      // [n_points_total][p][pk]: coefficient share w += weights[j][w][t] * A_j[t]
    std::vector<uint64_t> delta_tab;    // [m][p][pk]: row i >= 1 = w_{i-1} - w_i, row 0 = w_{m-1} (times the share of (-r)^t)
    std::vector<SpCluster> clusters;    // of the n-bit tree
    // variant bit 4 (DESIGN 14): the operator as a dense table of 2^n entries, T[u][w] = payload word w of the interval that
    // contains u, and its cyclic differences D[a][w] = T[(a-1) mod N][w] - T[a][w]
    std::vector<uint64_t> dense_t, dense_d;
    int atom_w[kMaxAtoms], atom_ib[kMaxAtoms], atom_ia[kMaxAtoms], alpha_atom[kMaxIntervals];
};

struct Program {
    // deep copy of the specification
    uint32_t n = 0, frac_bits = 0, m = 0, r = 0, d = 0, p_aux = 0, ell = 0, mask_output = 0, variant = 0;
    SpProgram sp;
    std::vector<uint64_t> alpha, coeff, aux;
    std::vector<fusefss_bitnode> nodes;
    std::vector<uint16_t> bit_root;
    std::vector<fusefss_kappa> kappa_a, kappa_b;
    std::vector<fusefss_phi_op> phi;
    // compiled shape
    uint64_t mask = 0;
    int M = 0, p = 0, Q = 0, T = 0, has_lut = 0;
    int n_carry = 0, n_kb = 0;
    int MA = 0, MB = 0, GMIX = 0, rounds = 0, n_out_a = 0, n_out_b = 0;
    int GA2B = 0, a2b_bit[kMaxA2B] = {0};   // A2B nodes with bit index j >= 1: one opened ring element + one j-bit bit-DCF key each (DESIGN 15)
    Atom atoms[kMaxAtoms];
    std::vector<Ins> ins;
    int n_areg = 0, n_breg = 0;
    int round_mul[kMaxRounds] = {0}, round_bits[kMaxRounds] = {0};
    // variant bit 1 (DESIGN 10): a product with the gate input x opens one ring element and needs (b, c = b r_in)
    uint32_t xmul = 0;
    uint32_t xpoly = 0;                   // variant bit 2 (DESIGN 11): Horner in the public xhat, zero Beaver rounds for the spline
    uint32_t dense = 0;                   // variant bit 4 (DESIGN 14): dense-table lookup by full-domain evaluation of the single key
    uint32_t et = 0;                      // variant bit 3 (DESIGN 13): bit trees stop max(k-7,0) levels deep, 128-bit leaf block
    int round_arr[kMaxRounds] = {0};      // ring-element arrays opened per round: 2 per Beaver, 1 per x-product
    int ma_is_x[64] = {0}, ma_word[65] = {0};
    // payload table v[i][w], i < m, w < p (coefficients poly-major, high degree first, then aux), masked
    std::vector<uint64_t> payload;
    // device copies of the small tables: one per device, uploaded on first use there (launchers), freed by fusefss_destroy.
    // The offsets inside the blob are fixed by compile_program.
    mutable std::mutex blob_mu;
    mutable std::map<int, void *> dev_blobs;
    size_t dev_ins_off = 0, dev_alpha_off = 0, dev_payload_off = 0, dev_blob_bytes = 0;
    size_t dev_sp_points_off = 0, dev_sp_weights_off = 0, dev_sp_delta_off = 0, dev_sp_clusters_off = 0;
    size_t dev_dense_t_off = 0, dev_dense_d_off = 0;
};

// 16-byte correction arrays of a bit tree on k input bits: k levels, or max(k-7,0) levels + the leaf block (DESIGN 13)
inline int bit_tree_levels(const Program &P, int k) { return P.et ? (k > 7 ? k - 7 : 0) : k; }
inline int bit_tree_arrays(const Program &P, int k) { return bit_tree_levels(P, k) + (P.et ? 1 : 0); }

int compile_program(const fusefss_spec *spec, Program **out);
void compute_layout(const Program &P, size_t count, Layout *L);
size_t post_msg_bytes(const Program &P, size_t count, int round);

}  // namespace fsk

struct fusefss_program { fsk::Program impl; };
