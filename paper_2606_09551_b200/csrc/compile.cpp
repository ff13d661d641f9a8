// compile.cpp -- fusefss_compile: operator specification -> compiled gate type (host only).
// Protocol 3 steps (2)-(4): normalise piecewise Boolean outputs with interval indicators
// (Lemma D.2), simplify descriptor-level sentinels, collect the primitive predicates in
// fixed descriptor order with spec-only dedup, rewrite each with the masked-comparison
// lemmas (Lemma 4.3, Lemma E.1, J.3 P:817-843), fix M = min(m+1, 2^n) and
// p = r(d+1) + p_aux, and lower Horner + the Boolean circuit + Phi (Def 4.2) into
// one straight-line program whose interactive gates are scheduled into rounds.  Format: DESIGN.md 4.3/4.6.
#include <algorithm>
#include <map>
#include <new>
#include <utility>

#include "program.h"

namespace fsk {
namespace {

uint64_t ring_mask(unsigned n) { return n >= 64 ? ~0ull : ((1ull << n) - 1ull); }

struct ViewRec { int k; uint64_t c; std::vector<uint64_t> betas; bool want_carry = false; };

// Builds the SSA program; registers are renamed to a small file afterwards.
class Lowering {
public:
    explicit Lowering(Program &prog) : P(prog) {}

    bool run();

private:
    Program &P;
    std::vector<ViewRec> views;
    std::vector<int> a_ready, b_ready;           // round at which an SSA value becomes available
    std::vector<int> node_val;                   // memo: bit node -> SSA bit value
    std::vector<int> calpha_val;                 // memo: C_{alpha_i} -> SSA bit value
    bool failed = false;
    int x_value = -1;                            // SSA value of x (Protocol 2)

    int view_index(int k, uint64_t c) {
        for (size_t v = 0; v < views.size(); ++v)
            if (views[v].k == k && views[v].c == c) return (int)v;
        views.push_back(ViewRec{k, c, {}, false});
        return (int)views.size() - 1;
    }
    void want_pred(int k, uint64_t c, uint64_t beta) {
        ViewRec &V = views[view_index(k, c)];
        if (std::find(V.betas.begin(), V.betas.end(), beta) == V.betas.end()) V.betas.push_back(beta);
    }
    int find_atom(int k, uint64_t c, bool theta, uint64_t beta) const {
        for (int t = 0; t < P.T; ++t) {
            const Atom &a = P.atoms[t];
            if (a.k == k && a.c == c && (a.is_theta != 0) == theta && (!theta || a.beta == beta)) return t;
        }
        return -1;
    }

    int fresh_a(int ready) { a_ready.push_back(ready); return (int)a_ready.size() - 1; }
    int fresh_b(int ready) { b_ready.push_back(ready); return (int)b_ready.size() - 1; }
    Ins &push(uint8_t op, int dst, int a, int b, uint64_t imm) {
        Ins i{};
        i.op = op; i.dst = (uint16_t)dst; i.a = (uint16_t)a; i.b = (uint16_t)b; i.imm = imm;
        P.ins.push_back(i);
        return P.ins.back();
    }

    // ---- bit values -------------------------------------------------------------------------
    int b_const(int v) { int d = fresh_b(0); push(I_B_CONST, d, 0, 0, (uint64_t)(v & 1)); return d; }
    int b_not(int a) { int d = fresh_b(b_ready[a]); push(I_B_NOT, d, a, 0, 0); return d; }
    int b_xor(int a, int b) { int d = fresh_b(std::max(b_ready[a], b_ready[b])); push(I_B_XOR, d, a, b, 0); return d; }
    int b_and(int a, int b) {                     // one Boolean AND gate = one bit triple, 2 opened bits
        int rd = std::max(b_ready[a], b_ready[b]);
        int d = fresh_b(rd + 1);
        Ins &i = push(I_B_AND, d, a, b, 0);
        i.gate = (uint16_t)P.MB++; i.round = (uint8_t)rd;
        if (rd >= kMaxRounds) failed = true;
        return d;
    }
    int b_or(int a, int b) { int na = b_not(a); int nb = b_not(b); return b_not(b_and(na, nb)); }
    // I[view_{k,c}(x) < beta] = A_theta xor A_r xor w   (Lemma 4.3 / E.1)
    int b_pred(int k, uint64_t c, uint64_t beta) {
        int at = find_atom(k, c, true, beta), ar = find_atom(k, c, false, 0);
        if (P.variant) { int v0 = fresh_b(0); push(I_B_ATOM, v0, at, 0, 0); return v0; }   // variant 1: the atom is the predicate share
        int v1 = fresh_b(0); push(I_B_ATOM, v1, at, 0, 0);
        int v2 = fresh_b(0); push(I_B_ATOM, v2, ar, 0, 0);
        int v3 = fresh_b(0); push(I_B_KAPPA, v3, P.atoms[at].carry, 0, 0);
        return b_xor(b_xor(v1, v2), v3);
    }
    int lower_bit(int id);
    int lower_boundary(int i);
    bool uniform_bit(uint32_t j) const {
        for (uint32_t i = 1; i < P.m; ++i)
            if (P.bit_root[(size_t)i * P.ell + j] != P.bit_root[j]) return false;
        return true;
    }
    // ---- arithmetic values ------------------------------------------------------------------
    int a_mul(int a, int b) {                     // one Beaver multiplication, 2 opened ring elements
        int rd = std::max(a_ready[a], a_ready[b]);
        int d = fresh_a(rd + 1);
        const bool ax = a == x_value, bx = b == x_value;
        const bool xm = P.xmul && ax != bx;       // variant bit 1: y * x with x = xhat - r_in, 1 opened element (DESIGN 10)
        Ins &i = xm ? push(I_A_MULX, d, ax ? b : a, 0, 0) : push(I_A_MUL, d, a, b, 0);
        i.gate = (uint16_t)P.MA++; i.round = (uint8_t)rd;
        if (rd >= kMaxRounds) failed = true;
        return d;
    }
    int a_bin(uint8_t op, int a, int b) { int d = fresh_a(std::max(a_ready[a], a_ready[b])); push(op, d, a, b, 0); return d; }

    void collect_atoms();
    void build_sp();
    bool lower_phi(int xval, const std::vector<int> &yval, const std::vector<int> &auxval, const std::vector<int> &zval);
    bool finish();
};

void Lowering::collect_atoms() {
    const int n = (int)P.n;
    for (const fusefss_bitnode &nd : P.nodes) {
        bool inner = !nd.value_is_2k && nd.value != 0;
        switch (nd.kind) {
        case FUSEFSS_BN_C: if (inner) want_pred(n, 0, nd.value); break;
        case FUSEFSS_BN_D: if (inner) want_pred(nd.k, 0, nd.value); break;
        case FUSEFSS_BN_MSB: want_pred(n, nd.value & P.mask, 1ull << (n - 1)); break;
        case FUSEFSS_BN_CARRY: views[view_index(nd.k, 0)].want_carry = true; break;
        default: break;
        }
    }
    bool piecewise = false;
    for (uint32_t j = 0; j < P.ell; ++j) piecewise = piecewise || !uniform_bit(j);
    if (piecewise || (P.variant && P.m > 1)) for (uint32_t i = 1; i < P.m; ++i) want_pred(n, 0, P.alpha[i - 1]);
    P.T = 0; P.n_carry = 0;
    for (const ViewRec &V : views) {
        if (P.T + 1 + (int)V.betas.size() > kMaxAtoms) { failed = true; return; }
        if (!P.variant || V.want_carry) P.atoms[P.T++] = Atom{V.k, V.c, 0, 0, -1};    // variant 1: r-atom only where CARRY reads it
        for (uint64_t beta : V.betas) P.atoms[P.T++] = Atom{V.k, V.c, 1, beta, P.variant ? -1 : P.n_carry++};
    }
    P.n_kb = P.n_carry + (int)P.kappa_b.size();
    if (P.n_kb > 64) failed = true;
    if (P.variant && !failed) build_sp();
}

// variant 1: evaluation points of the per-width keys, their linear contributions, and the prefix clusters.
// I[view_{k,c}(x) < beta] = e - b + a,  b = f(h), a = f(h - beta), h = (xhat + c) mod 2^k, f = I[. < r_k]  (DESIGN 9).
void Lowering::build_sp() {
    SpProgram &S = P.sp;
    S = SpProgram{};
    std::vector<std::vector<uint64_t>> deltas;
    auto width_of = [&](int k) {
        for (int w = 0; w < S.n_w; ++w) if (S.width[w].k == k) return w;
        if (S.n_w >= kMaxWidths) { failed = true; return 0; }
        S.width[S.n_w] = SpWidth{k, 0, 0, k == (int)P.n};
        deltas.emplace_back();
        return S.n_w++;
    };
    auto kmask = [](int k) { return k >= 64 ? ~0ull : ((1ull << k) - 1ull); };
    for (int t = 0; t < P.T; ++t) {
        const Atom &a = P.atoms[t];
        int w = width_of(a.k);
        if (failed) return;
        S.atom_w[t] = w;
        auto add = [&](uint64_t d) { if (std::find(deltas[w].begin(), deltas[w].end(), d) == deltas[w].end()) deltas[w].push_back(d); };
        add(a.c & kmask(a.k));
        if (a.is_theta) add((a.c - a.beta) & kmask(a.k));
    }
    int base = 0;
    for (int w = 0; w < S.n_w; ++w) {
        const uint64_t half = 1ull << (S.width[w].k - 1);
        std::sort(deltas[w].begin(), deltas[w].end(), [half](uint64_t x, uint64_t y) { return (x ^ half) < (y ^ half); });
        S.width[w].first_point = base; S.width[w].n_points = (int)deltas[w].size();
        for (uint64_t d : deltas[w]) S.points.push_back(SpPoint{d, 0});
        base += (int)deltas[w].size();
    }
    if (base > kMaxPoints) { failed = true; return; }
    auto index_of = [&](int w, uint64_t d) {
        for (int j = 0; j < S.width[w].n_points; ++j) if (S.points[S.width[w].first_point + j].delta == d) return j;
        return -1;
    };
    for (int t = 0; t < P.T; ++t) {
        const Atom &a = P.atoms[t];
        int w = S.atom_w[t];
        S.atom_ib[t] = index_of(w, a.c & kmask(a.k));
        S.atom_ia[t] = a.is_theta ? index_of(w, (a.c - a.beta) & kmask(a.k)) : -1;
        S.points[S.width[w].first_point + S.atom_ib[t]].bitmask ^= 1ull << t;      // LSB(e - b + a) = e ^ b ^ a
        if (a.is_theta) S.points[S.width[w].first_point + S.atom_ia[t]].bitmask ^= 1ull << t;
    }
    // interval lookup as a public linear map of the boundary comparisons (Lemma D.1 telescoped):
    // v_{i*} = v_{m-1} + sum_{i=1}^{m-1} (v_{i-1} - v_i) I[x < alpha_i]
    // With variant bit 2 the key's payload is (1, -r, .., (-r)^d) and the outputs are the coefficients of xhat^j of
    // P_{i*}(xhat - r): c'_j = sum_t sum_i J_i (-r)^t w_{i,j,t},  w_{i,j,t} = c_{i,j+t} C(j+t, j)  (DESIGN 11).
    const int p = P.p, d = (int)P.d, nc = (int)(P.r * (P.d + 1)), pk = P.xpoly ? d + 1 : 1;
    S.pk = pk;
    auto binom = [](int k, int j) { uint64_t v = 1; for (int i = 1; i <= j; ++i) v = v * (uint64_t)(k - j + i) / (uint64_t)i; return v; };
    auto wfun = [&](uint32_t i, int w, int t) -> uint64_t {
        if (!P.xpoly) return P.payload[(size_t)i * p + w];
        if (w >= nc) return t == 0 ? P.payload[(size_t)i * p + w] : 0;
        const int q = w / (d + 1), j = d - w % (d + 1);
        if (j + t > d) return 0;
        return (P.payload[(size_t)i * p + q * (d + 1) + (d - (j + t))] * binom(j + t, j)) & P.mask;
    };
    S.weights.assign((size_t)base * p * pk, 0);
    S.delta_tab.assign((size_t)P.m * p * pk, 0);
    for (int w = 0; w < p; ++w) for (int t = 0; t < pk; ++t) S.delta_tab[(size_t)w * pk + t] = wfun(P.m - 1, w, t);
    for (uint32_t i = 1; i < P.m && P.has_lut; ++i) {
        int ta = find_atom((int)P.n, 0, true, P.alpha[i - 1]);
        S.alpha_atom[i] = ta;
        const int wd = S.atom_w[ta];
        for (int w = 0; w < p; ++w) for (int t = 0; t < pk; ++t) {
            const uint64_t dl = (wfun(i - 1, w, t) - wfun(i, w, t)) & P.mask;
            S.delta_tab[((size_t)i * p + w) * pk + t] = dl;
            S.weights[((size_t)(S.width[wd].first_point + S.atom_ia[ta]) * p + w) * pk + t] += dl;
            S.weights[((size_t)(S.width[wd].first_point + S.atom_ib[ta]) * p + w) * pk + t] -= dl;
        }
    }
    // clusters of the n-bit tree: greedy over the sorted offsets; a cluster spans < 2^tail_bits, so its points have
    // at most two distinct (n - tail_bits)-bit prefixes; sharing must save at least 8 levels to be worth it
    for (int w = 0; w < S.n_w; ++w) {
        if (!S.width[w].is_vec) continue;
        const int n = (int)P.n, np = S.width[w].n_points, f0 = S.width[w].first_point;
        const uint64_t half = 1ull << (n - 1);
        int i = 0;
        while (i < np) {
            int j = i, bits = 0;
            while (j + 1 < np) {
                const uint64_t span = ((S.points[f0 + j + 1].delta ^ half) - (S.points[f0 + i].delta ^ half));
                int b = 0;
                while (b < 64 && (span >> b) != 0) ++b;                 // span < 2^b
                if (b > n - 8) break;
                bits = b; ++j;
            }
            S.clusters.push_back(SpCluster{i, j - i + 1, j > i ? (bits < 1 ? 1 : bits) : n, 0});
            i = j + 1;
        }
    }
}



int Lowering::lower_bit(int id) {
    if (id < 0 || id >= (int)P.nodes.size()) { failed = true; return b_const(0); }
    if (node_val[id] >= 0) return node_val[id];
    const fusefss_bitnode nd = P.nodes[id];
    const int n = (int)P.n;
    int v;
    switch (nd.kind) {
    case FUSEFSS_BN_CONST: v = b_const((int)(nd.value & 1)); break;
    case FUSEFSS_BN_C:
        v = nd.value_is_2k ? b_const(1) : nd.value == 0 ? b_const(0) : b_pred(n, 0, nd.value); break;
    case FUSEFSS_BN_D:
        v = nd.value_is_2k ? b_const(1) : nd.value == 0 ? b_const(0) : b_pred(nd.k, 0, nd.value); break;
    case FUSEFSS_BN_MSB:      // MSB(x+c) = not I[view_{n,c}(x) < 2^{n-1}]
        v = b_not(b_pred(n, nd.value & P.mask, 1ull << (n - 1))); break;
    case FUSEFSS_BN_CARRY:    // = the r-atom of view (k,0)  (DESIGN 4.3 R1)
        v = fresh_b(0); push(I_B_ATOM, v, find_atom(nd.k, 0, false, 0), 0, 0); break;
    case FUSEFSS_BN_NOT: v = b_not(lower_bit(nd.lhs)); break;
    case FUSEFSS_BN_XOR: { int a = lower_bit(nd.lhs); int b = lower_bit(nd.rhs); v = b_xor(a, b); break; }
    case FUSEFSS_BN_AND: { int a = lower_bit(nd.lhs); int b = lower_bit(nd.rhs); v = b_and(a, b); break; }
    case FUSEFSS_BN_OR:  { int a = lower_bit(nd.lhs); int b = lower_bit(nd.rhs); v = b_or(a, b); break; }
    default: failed = true; v = b_const(0);
    }
    node_val[id] = v;
    return v;
}

// C_{alpha_i}(x), i = 0..m, with the sentinels alpha_0 = 0 -> 0 and alpha_m = 2^n -> 1
int Lowering::lower_boundary(int i) {
    if (calpha_val[i] >= 0) return calpha_val[i];
    int v = i == 0 ? b_const(0) : i == (int)P.m ? b_const(1) : b_pred((int)P.n, 0, P.alpha[i - 1]);
    calpha_val[i] = v;
    return v;
}

bool Lowering::lower_phi(int xval, const std::vector<int> &yval, const std::vector<int> &auxval,
                         const std::vector<int> &zval) {
    std::vector<int> ua(256, -1), ub(256, -1);    // Phi's own registers -> SSA values
    auto A = [&](uint8_t r) { if (ua[r] < 0) failed = true; return ua[r] < 0 ? 0 : ua[r]; };
    auto B = [&](uint8_t r) { if (ub[r] < 0) failed = true; return ub[r] < 0 ? 0 : ub[r]; };
    for (const fusefss_phi_op &o : P.phi) {
        switch (o.op) {
        case FUSEFSS_PHI_A_CONST: { int d = fresh_a(0); push(I_A_CONST, d, 0, 0, o.imm & P.mask); ua[o.dst] = d; break; }
        case FUSEFSS_PHI_A_X: ua[o.dst] = xval; break;
        case FUSEFSS_PHI_A_Y: if (o.a >= yval.size()) return false; ua[o.dst] = yval[o.a]; break;
        case FUSEFSS_PHI_A_AUX: if (o.a >= auxval.size()) return false; ua[o.dst] = auxval[o.a]; break;
        case FUSEFSS_PHI_A_KAPPA: {
            if (o.a >= P.kappa_a.size()) return false;
            int d = fresh_a(0); push(I_A_KAPPA, d, o.a, 0, 0); ua[o.dst] = d; break; }
        case FUSEFSS_PHI_A_XHAT_SHR: { int d = fresh_a(0); push(I_A_XHAT_SHR, d, o.a, 0, 0); ua[o.dst] = d; break; }
        case FUSEFSS_PHI_A_ADD: { int a = A(o.a), b = A(o.b); ua[o.dst] = a_bin(I_A_ADD, a, b); break; }
        case FUSEFSS_PHI_A_SUB: { int a = A(o.a), b = A(o.b); ua[o.dst] = a_bin(I_A_SUB, a, b); break; }
        case FUSEFSS_PHI_A_MULC: { int a = A(o.a); int d = fresh_a(a_ready[a]); push(I_A_MULC, d, a, 0, o.imm); ua[o.dst] = d; break; }
        case FUSEFSS_PHI_A_MUL: { int a = A(o.a), b = A(o.b); ua[o.dst] = a_mul(a, b); break; }
        case FUSEFSS_PHI_A_B2A: {                 // one B2A gate: 1 opened bit
            int s = B(o.a), rd = b_ready[s];
            int d = fresh_a(rd + 1);
            Ins &i = push(I_A_B2A, d, s, 0, 0);
            i.gate = (uint16_t)P.GMIX++; i.round = (uint8_t)rd;
            if (rd >= kMaxRounds) failed = true;
            ua[o.dst] = d; break; }
        case FUSEFSS_PHI_A_OUT: if ((int)o.dst >= P.n_out_a) return false; push(I_A_OUT, o.dst, A(o.a), 0, 0); break;
        case FUSEFSS_PHI_B_CONST: ub[o.dst] = b_const((int)(o.imm & 1)); break;
        case FUSEFSS_PHI_B_Z: if (o.a >= zval.size()) return false; ub[o.dst] = zval[o.a]; break;
        case FUSEFSS_PHI_B_KAPPA: {
            if (o.a >= P.kappa_b.size()) return false;
            int d = fresh_b(0); push(I_B_KAPPA, d, P.n_carry + o.a, 0, 0); ub[o.dst] = d; break; }
        case FUSEFSS_PHI_B_XHAT: { int d = fresh_b(0); push(I_B_XHAT, d, o.a, 0, 0); ub[o.dst] = d; break; }
        case FUSEFSS_PHI_B_NOT: ub[o.dst] = b_not(B(o.a)); break;
        case FUSEFSS_PHI_B_XOR: { int a = B(o.a), b = B(o.b); ub[o.dst] = b_xor(a, b); break; }
        case FUSEFSS_PHI_B_AND: { int a = B(o.a), b = B(o.b); ub[o.dst] = b_and(a, b); break; }
        case FUSEFSS_PHI_B_OR: { int a = B(o.a), b = B(o.b); ub[o.dst] = b_or(a, b); break; }
        case FUSEFSS_PHI_B_ANDPUB: {
            int a = B(o.a); int d = fresh_b(b_ready[a]); push(I_B_ANDPUB, d, a, o.b, o.imm & 1); ub[o.dst] = d; break; }
        case FUSEFSS_PHI_B_OUT: if ((int)o.dst >= P.n_out_b || o.dst >= 64) return false; push(I_B_OUT, o.dst, B(o.a), 0, 0); break;
        case FUSEFSS_PHI_B_A2B: {                 // bit o.b of a shared ring element (DESIGN 15)
            if (o.b >= P.n) return false;
            const int s = A(o.a);
            if (failed) return false;
            if (o.b == 0) { int d = fresh_b(a_ready[s]); push(I_B_LSB, d, s, 0, 0); ub[o.dst] = d; break; }   // (e_0 + e_1) mod 2: local
            if (P.GA2B >= kMaxA2B) return false;
            const int rd = a_ready[s];
            int d = fresh_b(rd + 1);
            Ins &i = push(I_B_A2B, d, s, 0, (uint64_t)o.b);
            P.a2b_bit[P.GA2B] = (int)o.b; i.gate = (uint16_t)P.GA2B++; i.round = (uint8_t)rd;
            if (rd >= kMaxRounds) failed = true;
            ub[o.dst] = d; break; }
        default: return false;
        }
        if (failed) return false;
    }
    return true;
}

bool Lowering::run() {
    collect_atoms();
    if (failed) return false;
    node_val.assign(P.nodes.size(), -1);
    calpha_val.assign(P.m + 1, -1);
    const uint32_t per_poly = P.d + 1, n_coeff = P.r * per_poly;

    int xval = fresh_a(0); push(I_A_X, xval, 0, 0, 0);
    x_value = xval;                       // Protocol 2
    std::vector<int> cval(P.p);
    for (int w = 0; w < P.p; ++w) {
        cval[w] = fresh_a(0);
        if (P.has_lut) push(I_A_COEFF, cval[w], w, 0, 0);
        else push(I_A_CONST, cval[w], 0, 0, P.payload[w]);                   // m = 1: public descriptor constants
    }
    std::vector<int> yval(P.r), auxval(P.p_aux), zval(P.ell);
    for (uint32_t j = 0; j < P.r; ++j) yval[j] = cval[j * per_poly];
    for (uint32_t k = 1; k <= P.d; ++k)                                      // Horner, one round per step
        for (uint32_t j = 0; j < P.r; ++j) {
            if (P.xpoly) {                                                   // (..(c'_d xhat + c'_{d-1}) xhat ..) + c'_0, local (DESIGN 11)
                int pr = fresh_a(a_ready[yval[j]]);
                push(I_A_MULXH, pr, yval[j], 0, 0);
                yval[j] = a_bin(I_A_ADD, pr, cval[j * per_poly + k]);
                continue;
            }
            int prod = a_mul(yval[j], xval);
            yval[j] = a_bin(I_A_ADD, prod, cval[j * per_poly + k]);
        }
    for (uint32_t j = 0; j < P.p_aux; ++j) auxval[j] = cval[n_coeff + j];
    for (uint32_t j = 0; j < P.ell; ++j) {
        if (uniform_bit(j)) { zval[j] = lower_bit(P.bit_root[j]); continue; }
        int acc = -1;                                                        // XOR_i (J_i and B_i)  (Lemma D.2)
        for (uint32_t i = 0; i < P.m; ++i) {
            int hi = lower_boundary((int)i + 1), lo = lower_boundary((int)i);
            int J = b_xor(hi, lo);                                           // Lemma D.1
            int Bi = lower_bit(P.bit_root[(size_t)i * P.ell + j]);
            int term = b_and(J, Bi);
            acc = acc < 0 ? term : b_xor(acc, term);
        }
        zval[j] = acc;
    }
    if (failed) return false;
    if (P.phi.empty()) {
        P.n_out_a = (int)P.r; P.n_out_b = (int)P.ell;
        for (uint32_t j = 0; j < P.r; ++j) push(I_A_OUT, (int)j, yval[j], 0, 0);
        for (uint32_t j = 0; j < P.ell; ++j) push(I_B_OUT, (int)j, zval[j], 0, 0);
    } else if (!lower_phi(xval, yval, auxval, zval)) return false;
    return finish();
}

// Message positions per round, round count, and renaming of SSA values onto a small register file
// (a value's register is released after its last use; interactive results keep theirs).
bool Lowering::finish() {
    if (failed) return false;
    P.rounds = 0;
    int mulpos[kMaxRounds] = {0}, bitpos[kMaxRounds] = {0};
    for (Ins &i : P.ins) {
        if (i.op == I_A_MUL || i.op == I_A_MULX) {
            const int arrs = i.op == I_A_MUL ? 2 : 1;
            i.pos = (uint16_t)mulpos[i.round]; mulpos[i.round] += arrs;           // pos = first opened array of the gate in its round
            P.round_mul[i.round]++;
            P.ma_is_x[i.gate] = i.op == I_A_MULX;
            P.rounds = std::max(P.rounds, i.round + 1);
        }
        else if (i.op == I_B_A2B) { i.pos = (uint16_t)mulpos[i.round]; mulpos[i.round] += 1; P.rounds = std::max(P.rounds, i.round + 1); }
        else if (i.op == I_B_AND) { i.pos = (uint16_t)bitpos[i.round]; bitpos[i.round] += 2; P.rounds = std::max(P.rounds, i.round + 1); }
        else if (i.op == I_A_B2A) { i.pos = (uint16_t)bitpos[i.round]; bitpos[i.round] += 1; P.rounds = std::max(P.rounds, i.round + 1); }
    }
    if (P.rounds > kMaxRounds || P.MB > 64 || P.GMIX > 64 || P.MA > 64) return false;
    for (int g = 0; g < P.MA; ++g) P.ma_word[g + 1] = P.ma_word[g] + (P.ma_is_x[g] ? 2 : 3);
    for (Ins &i : P.ins) if (i.op == I_A_MUL || i.op == I_A_MULX) i.imm = (uint64_t)P.ma_word[i.gate];
    for (int q = 0; q < kMaxRounds; ++q) {
        P.round_arr[q] = mulpos[q]; P.round_bits[q] = bitpos[q];
        if (bitpos[q] > 64) return false;
    }
    // last use of every SSA value
    const int NI = (int)P.ins.size();
    std::vector<int> a_last(a_ready.size(), -1), b_last(b_ready.size(), -1);
    auto reads = [](const Ins &i, bool &a_is_A, bool &a_is_B, bool &b_is_A, bool &b_is_B) {
        a_is_A = a_is_B = b_is_A = b_is_B = false;
        switch (i.op) {
        case I_B_NOT: case I_B_ANDPUB: case I_B_OUT: case I_A_B2A: a_is_B = true; break;
        case I_B_XOR: case I_B_AND: a_is_B = b_is_B = true; break;
        case I_A_ADD: case I_A_SUB: case I_A_MUL: a_is_A = b_is_A = true; break;
        case I_A_MULC: case I_A_OUT: case I_A_MULX: case I_A_MULXH: case I_B_LSB: case I_B_A2B: a_is_A = true; break;
        default: break;
        }
    };
    for (int t = 0; t < NI; ++t) {
        bool aA, aB, bA, bB; reads(P.ins[t], aA, aB, bA, bB);
        if (aA) a_last[P.ins[t].a] = t;
        if (aB) b_last[P.ins[t].a] = t;
        if (bA) a_last[P.ins[t].b] = t;
        if (bB) b_last[P.ins[t].b] = t;
    }
    std::vector<int> a_map(a_ready.size(), -1), b_map(b_ready.size(), -1), a_free, b_free;
    int a_next = 0, b_next = 0;
    auto writes_a = [](uint8_t op) { return op >= I_A_CONST && op <= I_A_B2A; };
    auto writes_b = [](uint8_t op) { return (op >= I_B_CONST && op <= I_B_ANDPUB) || op == I_B_LSB || op == I_B_A2B; };
    for (int t = 0; t < NI; ++t) {
        Ins &i = P.ins[t];
        bool aA, aB, bA, bB; reads(i, aA, aB, bA, bB);
        int sa = i.a, sb = i.b;
        if (aA) i.a = (uint16_t)a_map[sa];
        if (aB) i.a = (uint16_t)b_map[sa];
        if (bA) i.b = (uint16_t)a_map[sb];
        if (bB) i.b = (uint16_t)b_map[sb];
        // release sources whose last use is here (before allocating dst, so dst may reuse them)
        if (aA && a_last[sa] == t) a_free.push_back(a_map[sa]);
        if (bA && a_last[sb] == t && sb != sa) a_free.push_back(a_map[sb]);
        if (aB && b_last[sa] == t) b_free.push_back(b_map[sa]);
        if (bB && b_last[sb] == t && sb != sa) b_free.push_back(b_map[sb]);
        if (writes_a(i.op)) {
            int ssa = i.dst, reg;
            if (!a_free.empty()) { reg = a_free.back(); a_free.pop_back(); } else reg = a_next++;
            a_map[ssa] = reg; i.dst = (uint16_t)reg;
            if (a_last[ssa] < 0) a_free.push_back(reg);                      // dead value
        } else if (writes_b(i.op)) {
            int ssa = i.dst, reg;
            if (!b_free.empty()) { reg = b_free.back(); b_free.pop_back(); } else reg = b_next++;
            b_map[ssa] = reg; i.dst = (uint16_t)reg;
            if (b_last[ssa] < 0) b_free.push_back(reg);
        }
    }
    P.n_areg = a_next; P.n_breg = b_next;
    return a_next <= kMaxAReg && b_next <= kMaxBReg;
}

}  // namespace

int compile_program(const fusefss_spec *S, Program **out) {
    if (!S || !out) return FUSEFSS_E_NULL;
    *out = nullptr;
    if (S->n < 1 || S->n > 64 || S->m < 1 || S->m >= (uint32_t)kMaxIntervals) return FUSEFSS_E_SPEC;
    if (S->r > (uint32_t)kMaxP || S->d > (uint32_t)kMaxP || S->p_aux > (uint32_t)kMaxP || S->ell > 64) return FUSEFSS_E_SPEC;
    const uint32_t per_poly = S->d + 1, n_coeff = S->r * per_poly, p = n_coeff + S->p_aux;
    if (p < 1 || p > (uint32_t)kMaxP) return FUSEFSS_E_SPEC;
    if ((S->m > 1 && !S->alpha) || (n_coeff && !S->coeff) || (S->p_aux && !S->aux) || (S->n_nodes && !S->nodes) ||
        (S->ell && !S->bit_root) || (S->n_kappa_a && !S->kappa_a) || (S->n_kappa_b && !S->kappa_b) ||
        (S->phi_len && !S->phi))
        return FUSEFSS_E_NULL;
    const uint64_t mask = ring_mask(S->n);
    for (uint32_t i = 0; i + 1 < S->m; ++i) {     // well-formedness: 0 < alpha_1 < ... < alpha_{m-1} < 2^n
        if (S->alpha[i] == 0 || (S->alpha[i] & ~mask)) return FUSEFSS_E_SPEC;
        if (i && S->alpha[i] <= S->alpha[i - 1]) return FUSEFSS_E_SPEC;
    }
    for (uint32_t i = 0; i < S->n_nodes; ++i) {
        const fusefss_bitnode &nd = S->nodes[i];
        if (nd.kind > FUSEFSS_BN_OR) return FUSEFSS_E_SPEC;
        if ((nd.kind == FUSEFSS_BN_D || nd.kind == FUSEFSS_BN_CARRY) && (nd.k < 1 || nd.k > S->n)) return FUSEFSS_E_SPEC;
        if (nd.kind >= FUSEFSS_BN_NOT && nd.lhs >= i) return FUSEFSS_E_SPEC;                 // DAG: operands precede
        if (nd.kind >= FUSEFSS_BN_XOR && nd.rhs >= i) return FUSEFSS_E_SPEC;
    }
    for (size_t i = 0; i < (size_t)S->m * S->ell; ++i) if (S->bit_root[i] >= S->n_nodes) return FUSEFSS_E_SPEC;
    for (uint32_t i = 0; i < S->n_nodes; ++i) {   // values in range: beta in [0, 2^n] / gamma in [0, 2^k] (the upper ends via value_is_2k)
        const fusefss_bitnode &nd = S->nodes[i];
        if (nd.kind == FUSEFSS_BN_C && !nd.value_is_2k && (nd.value & ~mask)) return FUSEFSS_E_SPEC;
        if (nd.kind == FUSEFSS_BN_D && !nd.value_is_2k && (nd.value & ~ring_mask(nd.k))) return FUSEFSS_E_SPEC;
    }
    if (S->n_kappa_a > 8 || S->n_kappa_b > 64) return FUSEFSS_E_SPEC;
    for (uint32_t i = 0; i < S->n_kappa_a; ++i)
        if (S->kappa_a[i].kind != FUSEFSS_KA_R_SHR || S->kappa_a[i].arg >= 64) return FUSEFSS_E_SPEC;
    for (uint32_t i = 0; i < S->n_kappa_b; ++i)
        if (S->kappa_b[i].kind != FUSEFSS_KB_R_BIT || S->kappa_b[i].arg >= S->n) return FUSEFSS_E_SPEC;
    if (S->phi_len) {                             // Phi: public bit indices below n, every declared output written exactly once
        uint32_t wa[256] = {0}, wb[256] = {0};
        for (uint32_t i = 0; i < S->phi_len; ++i) {
            const fusefss_phi_op &o = S->phi[i];
            if (o.op == FUSEFSS_PHI_B_XHAT && o.a >= S->n) return FUSEFSS_E_SPEC;
            if (o.op == FUSEFSS_PHI_B_ANDPUB && o.b >= S->n) return FUSEFSS_E_SPEC;
            if (o.op == FUSEFSS_PHI_A_XHAT_SHR && o.a > 64) return FUSEFSS_E_SPEC;
            if (o.op == FUSEFSS_PHI_A_OUT) ++wa[o.dst];
            if (o.op == FUSEFSS_PHI_B_OUT) ++wb[o.dst];
        }
        for (uint32_t j = 0; j < 256; ++j) {
            if (wa[j] != (j < S->n_out_a ? 1u : 0u)) return FUSEFSS_E_SPEC;
            if (wb[j] != (j < S->n_out_b ? 1u : 0u)) return FUSEFSS_E_SPEC;
        }
    }

    fusefss_program *holder = new (std::nothrow) fusefss_program();
    if (!holder) return FUSEFSS_E_SPEC;
    Program &P = holder->impl;
    P.n = S->n; P.frac_bits = S->frac_bits; P.m = S->m; P.r = S->r; P.d = S->d; P.p_aux = S->p_aux; P.ell = S->ell;
    P.mask_output = S->mask_output ? 1 : 0;
    P.mask = mask;
    if (S->m > 1) P.alpha.assign(S->alpha, S->alpha + (S->m - 1));
    if (n_coeff) P.coeff.assign(S->coeff, S->coeff + (size_t)S->m * n_coeff);
    if (S->p_aux) P.aux.assign(S->aux, S->aux + (size_t)S->m * S->p_aux);
    if (S->n_nodes) P.nodes.assign(S->nodes, S->nodes + S->n_nodes);
    if (S->ell) P.bit_root.assign(S->bit_root, S->bit_root + (size_t)S->m * S->ell);
    if (S->n_kappa_a) P.kappa_a.assign(S->kappa_a, S->kappa_a + S->n_kappa_a);
    if (S->n_kappa_b) P.kappa_b.assign(S->kappa_b, S->kappa_b + S->n_kappa_b);
    if (S->phi_len) P.phi.assign(S->phi, S->phi + S->phi_len);
    P.p = (int)p; P.Q = ((int)p + 1) / 2;
    // M = min(m+1, 2^n)  (Protocol 3 line 2)
    P.M = (S->n >= 7 || (uint64_t)(S->m + 1) < (1ull << S->n)) ? (int)S->m + 1 : (int)(1ull << S->n);
    P.has_lut = S->m > 1;                         // a single interval needs no lookup
    P.variant = S->variant & 1;
    P.xmul = (S->variant >> 1) & 1;
    P.xpoly = ((S->variant >> 2) & 1) && S->d >= 1 && S->m > 1;
    P.et = (S->variant >> 3) & 1;
    P.dense = (S->variant >> 4) & 1;
    if (P.dense && (!P.variant || P.xpoly || S->n > 16)) { delete holder; return FUSEFSS_E_SPEC; }   // needs the single key, n <= 16
    if (P.xpoly && S->d > 2) { delete holder; return FUSEFSS_E_SPEC; }          // kernels are instantiated for d <= 2
    if (P.variant) P.M = (int)S->m;               // variant 1: no translated partition, no wrap / dummy split
    P.n_out_a = (int)S->n_out_a; P.n_out_b = (int)S->n_out_b;
    if (P.n_out_a > kMaxP || P.n_out_b > 64) { delete holder; return FUSEFSS_E_SPEC; }
    P.payload.resize((size_t)S->m * p);
    for (uint32_t i = 0; i < S->m; ++i) {
        for (uint32_t q = 0; q < n_coeff; ++q) P.payload[(size_t)i * p + q] = P.coeff[(size_t)i * n_coeff + q] & mask;
        for (uint32_t q = 0; q < S->p_aux; ++q) P.payload[(size_t)i * p + n_coeff + q] = P.aux[(size_t)i * S->p_aux + q] & mask;
    }
    Lowering low(P);
    if (!low.run()) { delete holder; return FUSEFSS_E_SPEC; }
    if (P.dense && P.has_lut) {                  // the operator as a table of 2^n entries and its cyclic differences (DESIGN 14)
        const size_t N = (size_t)1 << P.n, pp = (size_t)P.p;
        P.sp.dense_t.resize(N * pp);
        P.sp.dense_d.resize(N * pp);
        size_t i = 0;
        for (size_t u = 0; u < N; ++u) {
            while (i + 1 < P.m && u >= P.alpha[i]) ++i;
            for (size_t w = 0; w < pp; ++w) P.sp.dense_t[u * pp + w] = P.payload[i * pp + w];
        }
        for (size_t a = 0; a < N; ++a)
            for (size_t w = 0; w < pp; ++w)
                P.sp.dense_d[a * pp + w] = (P.sp.dense_t[((a + N - 1) % N) * pp + w] - P.sp.dense_t[a * pp + w]) & P.mask;
    }
    {   // layout of the small device tables (uploaded per device on first use)
        auto up = [](size_t x) { return (x + 255) & ~(size_t)255; };
        P.dev_ins_off = 0;
        P.dev_alpha_off = up(P.ins.size() * sizeof(Ins));
        P.dev_payload_off = P.dev_alpha_off + up(P.alpha.size() * 8 + 8);
        P.dev_sp_points_off = P.dev_payload_off + up(P.payload.size() * 8 + 8);
        P.dev_sp_weights_off = P.dev_sp_points_off + up(P.sp.points.size() * sizeof(SpPoint) + 8);
        P.dev_sp_delta_off = P.dev_sp_weights_off + up(P.sp.weights.size() * 8 + 8);
        P.dev_sp_clusters_off = P.dev_sp_delta_off + up(P.sp.delta_tab.size() * 8 + 8);
        P.dev_dense_t_off = P.dev_sp_clusters_off + up(P.sp.clusters.size() * sizeof(SpCluster) + 8);
        P.dev_dense_d_off = P.dev_dense_t_off + up(P.sp.dense_t.size() * 8 + 8);
        P.dev_blob_bytes = P.dev_dense_d_off + up(P.sp.dense_d.size() * 8 + 8);
    }
    *out = &holder->impl;
    return FUSEFSS_OK;
}

static size_t round_up_256(size_t x) { return (x + 255) & ~(size_t)255; }

void compute_layout(const Program &P, size_t count, Layout *L) {
    size_t off = 0;
    L->s16 = round_up_256(count * 16);
    L->s8 = round_up_256(count * 8);
    if (P.variant) {                              // one tree per view width (DESIGN 9)
        L->lvl_stride = L->s16 + (size_t)P.sp.pk * L->s8;
        L->vt_lvl_rel = L->s16;
        L->vt_fin_rel = L->s16 + L->lvl_stride * (size_t)P.n;
        L->vt_stride = L->vt_fin_rel + (size_t)P.sp.pk * L->s8;
        L->lut_c = L->vt_first = 0;
        for (int w = 0; w < P.sp.n_w; ++w) {
            if (!P.sp.width[w].is_vec) {
                L->bt_root[w] = off; off += L->s16;
                L->bt_cw[w] = off;   off += L->s16 * (size_t)bit_tree_arrays(P, P.sp.width[w].k);
                L->bt_vb[w] = off;   off += L->s8;
            } else { L->vt_first = off; off += L->vt_stride; }
        }
    }
    for (int t = 0; t < P.T && !P.variant; ++t) {
        L->bt_root[t] = off; off += L->s16;
        L->bt_cw[t] = off;   off += L->s16 * (size_t)bit_tree_arrays(P, P.atoms[t].k);
        L->bt_vb[t] = off;   off += L->s8;
    }
    const size_t pw = (size_t)P.p * L->s8;
    if (!P.variant) {
        L->lvl_stride = L->s16 + pw;
        L->vt_lvl_rel = L->s16;                               // after the root
        L->vt_fin_rel = L->s16 + L->lvl_stride * (size_t)P.n;
        L->vt_stride = L->vt_fin_rel + pw;
        L->lut_c = off; L->vt_first = off;
    }
    if (P.has_lut && !P.variant) {
        off += pw;
        L->vt_first = off;
        off += L->vt_stride * (size_t)(P.M - 1);
    }
    L->rin = off;      off += L->s8;
    L->rout = off;     if (P.mask_output) off += (size_t)P.n_out_a * L->s8;
    L->ka = off;       off += P.kappa_a.size() * L->s8;
    L->rpow = off;     if (P.variant && P.xpoly) off += (size_t)P.d * L->s8;        // shares of (-r)^t, t = 1..d
    L->kb = off;       if (P.n_kb > 0) off += L->s8;
    L->beaver = off;   off += (size_t)P.ma_word[P.MA] * L->s8;
    L->andt = off;     if (P.MB > 0) off += 3 * L->s8;
    L->b2a_bits = off; if (P.GMIX > 0) off += L->s8;
    L->b2a_a = off;    off += (size_t)P.GMIX * L->s8;
    L->a2b_rho = off;  off += (size_t)P.GA2B * L->s8;                             // [rho_i], one word of <bit_j(rho_i)>, then one
    L->a2b_bits = off; if (P.GA2B > 0) off += L->s8;                              // j_i-bit comparison key per node (DESIGN 15)
    for (int i = 0; i < P.GA2B; ++i) {
        L->a2b_root[i] = off; off += L->s16;
        L->a2b_cw[i] = off;   off += L->s16 * (size_t)bit_tree_arrays(P, P.a2b_bit[i]);
        L->a2b_vb[i] = off;   off += L->s8;
    }
    L->total = off;
}

size_t post_msg_bytes(const Program &P, size_t count, int round) {
    if (round < 0 || round >= P.rounds) return 0;
    return round_up_256(count * 8) * ((size_t)P.round_arr[round] + (P.round_bits[round] ? 1 : 0));
}

}  // namespace fsk
