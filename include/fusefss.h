/*
 * fusefss.h -- C ABI of libfusefss (B200 / sm_100a), the data-parallel hot path of FuseFSS
 * (arxiv/paper_2606_09551).  "P:<line>" cites /root/reference/PAPER.md; "DESIGN 4.x" cites DESIGN.md.
 *
 * Conventions
 *  - Every function returns 0 on success or a negative FUSEFSS_E_* code; nothing throws or aborts.
 *    fusefss_strerror() gives text.  Size queries return 0 on a null program.
 *  - Ring elements of Z_{2^n} (n <= 64) travel as uint64_t with bits >= n zero.
 *  - Pointers named *_dev are DEVICE pointers owned by the caller (e.g. torch tensors); pointers without
 *    the suffix are HOST pointers.  The library allocates no device memory of its own except one small buffer per
 *    (program, device): its post-processing code and descriptor tables -- a few KB; for dense-table programs (variant bit 4) also the
 *    2 x 2^n x p x 8-byte table, 2 MB at n = 16, p = 2.  fusefss_prepare() uploads it; otherwise the first call that needs it does
 *    (one cudaMalloc + one synchronous cudaMemcpy, so call fusefss_prepare at start-up if first-use stalls matter).  Freed by _destroy.
 *    fusefss_post_fused_noalloc needs no such buffer at all.
 *  - `stream` is a cudaStream_t passed as void* (NULL = default stream); once a program is prepared all launches are asynchronous on it.
 *  - party is 0 or 1.  xhat = x + r_in mod 2^n is public and identical for both parties (Protocol 1).
 *  - A key buffer is one-time material for exactly one xhat tensor; not enforced.
 *  - Key buffers are SoA over the chunk's elements; their size and layout depend on (program, count) only
 *    (Prop. I.3; DESIGN 4.4).
 */
#ifndef FUSEFSS_H
#define FUSEFSS_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum {
    FUSEFSS_OK = 0,
    FUSEFSS_E_NULL = -1,      /* a required pointer is null                                   */
    FUSEFSS_E_SPEC = -2,      /* ill-formed operator specification or over a limit    */
    FUSEFSS_E_PARTY = -3,     /* party not in {0,1}                                           */
    FUSEFSS_E_COUNT = -4,     /* count == 0                                                   */
    FUSEFSS_E_ROUND = -5,     /* round outside [0, rounds]                                    */
    FUSEFSS_E_CUDA = -6,      /* a CUDA call failed (fusefss_last_cuda_error() has the text)  */
    FUSEFSS_E_OMITTED = -7,   /* eval_cmp with T = 0 / eval_lut with m = 1 (call omitted) */
    FUSEFSS_E_WORKSPACE = -8, /* fusefss_gate_host: workspace_bytes < fusefss_gate_workspace_bytes()  */
    FUSEFSS_E_DEBUG = -9,     /* fusefss_debug_set: unknown knob                                      */
    FUSEFSS_E_STATIC = -10    /* fusefss_post_fused_noalloc: the lowered program has more than FUSEFSS_NOALLOC_MAX_INS instructions */
};

/* ---- operator specification (Def 4.1; grammar App. H) ------------------ */
/* Boolean expression DAG node.  kind: */
enum { FUSEFSS_BN_CONST = 0,   /* value & 1                                                     */
       FUSEFSS_BN_C = 1,       /* C_beta(x)    = I[rep(x) < value]; value_is_2k: beta = 2^n     */
       FUSEFSS_BN_D = 2,       /* D_{gamma,k}(x) = I[(rep(x) mod 2^k) < value]; value_is_2k: 2^k */
       FUSEFSS_BN_MSB = 3,     /* MSB(x + value)                                   */
       FUSEFSS_BN_CARRY = 4,   /* carry of the low k bits of x + r_in (DESIGN 4.3 R1)           */
       FUSEFSS_BN_NOT = 5, FUSEFSS_BN_XOR = 6, FUSEFSS_BN_AND = 7, FUSEFSS_BN_OR = 8 };
typedef struct {
    uint8_t kind, k; uint16_t lhs, rhs; uint8_t value_is_2k, pad; uint64_t value;
} fusefss_bitnode;

/* instance constants kappa derived from r_in only (Def 4.2) */
enum { FUSEFSS_KA_R_SHR = 1 /* kappa^A = rep(r_in) >> arg */, FUSEFSS_KB_R_BIT = 2 /* kappa^B = bit arg of r_in */ };
typedef struct { uint8_t kind, arg; } fusefss_kappa;

/* post-processing program Phi (App. H): straight-line code over arithmetic registers A[]
 * and bit registers B[] (at most 256 of each).  op: */
enum {
    FUSEFSS_PHI_A_CONST = 1,  /* A[dst] = imm                        */
    FUSEFSS_PHI_A_X,          /* A[dst] = x                          */
    FUSEFSS_PHI_A_Y,          /* A[dst] = y_a (a-th polynomial)      */
    FUSEFSS_PHI_A_KAPPA,      /* A[dst] = kappa^A_a                  */
    FUSEFSS_PHI_A_XHAT_SHR,   /* A[dst] = xhat >> a   (public)       */
    FUSEFSS_PHI_A_ADD, FUSEFSS_PHI_A_SUB,     /* A[dst] = A[a] +- A[b] */
    FUSEFSS_PHI_A_MULC,       /* A[dst] = A[a] * imm                 */
    FUSEFSS_PHI_A_MUL,        /* A[dst] = A[a] * A[b]  (one Beaver)  */
    FUSEFSS_PHI_A_B2A,        /* A[dst] = B[a]         (one B2A)     */
    FUSEFSS_PHI_A_OUT,        /* output y'[dst] = A[a]               */
    FUSEFSS_PHI_A_AUX,        /* A[dst] = aux_a of the active interval */
    FUSEFSS_PHI_B_CONST = 32, /* B[dst] = imm & 1                    */
    FUSEFSS_PHI_B_Z,          /* B[dst] = z_a (a-th predicate bit)   */
    FUSEFSS_PHI_B_KAPPA,      /* B[dst] = kappa^B_a                  */
    FUSEFSS_PHI_B_XHAT,       /* B[dst] = bit a of xhat (public)     */
    FUSEFSS_PHI_B_NOT, FUSEFSS_PHI_B_XOR, FUSEFSS_PHI_B_AND, FUSEFSS_PHI_B_OR,
    FUSEFSS_PHI_B_ANDPUB,     /* B[dst] = B[a] & (bit b of xhat ^ (imm&1)) */
    FUSEFSS_PHI_B_OUT,        /* output z'[dst] = B[a]               */
    FUSEFSS_PHI_B_A2B         /* B[dst] = bit b of the ring element A[a]: the A2B node ([x] -> <b> "for a suitable extracted bit b",
                                 P:81, 683-685).  b = 0 is local (XOR of the shares' low bits); b >= 1 costs one opened ring
                                 element and one b-bit comparison key from the dealer, one round (DESIGN 15); at most 8 per gate */
};
typedef struct { uint8_t op, dst, a, b; uint32_t pad; uint64_t imm; } fusefss_phi_op;

typedef struct {
    uint32_t n, frac_bits;            /* ring Z_{2^n}, fixed-point metadata                         */
    uint32_t m, r, d, p_aux, ell;     /* intervals, polynomials, degree bound, aux constants, predicate bits */
    uint32_t n_nodes, n_kappa_a, n_kappa_b, phi_len;
    uint32_t n_out_a, n_out_b;        /* outputs of Phi (ignored when phi_len == 0: outputs are y and z)    */
    uint32_t mask_output;             /* 1: arithmetic outputs are opened as yhat = y + r_out       */
    uint32_t variant;                 /* bit 0: single-key shared-prefix construction (DESIGN 9); bit 1: input-masked products
                                         (DESIGN 10); bit 2: Horner in the public xhat (DESIGN 11); bit 3: early-terminated bit trees
                                         (DESIGN 13); bit 4: dense-table lookup by full-domain evaluation, needs bit 0 and n <= 16
                                         (DESIGN 14).  0 = the paper's Protocol 3 with textbook subprotocols. */
    const uint64_t *alpha;            /* HOST [m-1] interior boundaries, strictly increasing in (0, 2^n)    */
    const uint64_t *coeff;            /* HOST [m][r][d+1], high degree first                                */
    const uint64_t *aux;              /* HOST [m][p_aux]                                                    */
    const fusefss_bitnode *nodes;     /* HOST [n_nodes]                                                     */
    const uint16_t *bit_root;         /* HOST [m][ell] root node per interval per output bit                */
    const fusefss_kappa *kappa_a, *kappa_b;
    const fusefss_phi_op *phi;        /* HOST [phi_len]                                                     */
} fusefss_spec;

typedef struct fusefss_program fusefss_program;   /* opaque, library-owned */

/* L_shape = (T, {k_t}, M, p, #mults, #ANDs, #mixed-domain conversions) -- everything that may depend on the spec only
 * (P:195, 905-909); G_mix counts B2A and (interactive) A2B conversions */
typedef struct {
    int32_t T, M, p, M_A, M_B, G_mix, rounds, n_out_a, n_out_b, has_lut, n_kb;
    int32_t k[64];
} fusefss_shape_t;

/* ---- a0: compile (host only; Protocol 3 steps (2)-(4); DESIGN 4.3) ------------------
 * Validates the spec (boundaries strictly increasing in (0,2^n), n in [1,64], m < 64, p <= 8, T <= 64,
 * <= 16 rounds, <= 64 AND gates, <= 64 B2A gates, <= 8 interactive A2B nodes, <= 64 opened bits per round -- an AND opens 2, a B2A 1 --,
 * <= 48 live arithmetic and <= 128 live bit values) and builds the immutable compiled gate type: atom list,
 * (T, M, p), post-processing program, message shapes.  The spec's arrays are copied; the caller may free
 * them.  Compile once per gate type, reuse across tensors/layers (program caching). */
int fusefss_compile(const fusefss_spec *spec, fusefss_program **out);
void fusefss_destroy(fusefss_program *prog);
/* Uploads the program's device tables to the CURRENT device now (see Conventions) and initialises the library's per-device constants
 * (PRG round keys and T-table seed in constant memory).  Idempotent and optional; after it no keygen / eval / post call with this program
 * on this device allocates device memory or synchronises the device. */
int fusefss_prepare(const fusefss_program *prog);
int fusefss_shape(const fusefss_program *prog, fusefss_shape_t *out);
/* atom t of the packed comparison instance Q = ((k_t, c_t, theta_t)) (Def I.1):
 * out4 = { k_t, c_t, is_theta, beta_t };  theta_t = (r mod 2^k + beta_t) mod 2^k, or r mod 2^k for an r-atom */
int fusefss_atom(const fusefss_program *prog, int t, uint64_t *out4);
/* bytes of ONE party's key buffer for `count` elements (DESIGN 4.4); a function of (program, count) only */
size_t fusefss_key_bytes(const fusefss_program *prog, size_t count);

/* ---- a1-a4: keygen (dealer; section 5.2; Protocol 3 steps (1),(5)) ----
 * r_in_dev[count]: fresh uniform input masks; r_out_dev[n_out_a][count]: output masks (may be NULL unless
 * mask_output).  seed: the dealer's randomness seed (DESIGN 4.5) -- a reproducibility handle with 64 bits of entropy, one per
 * gate instance; a deployment draws the dealer's 128-bit AES key from a CSPRNG instead.  first_elem: GLOBAL index of element 0 of
 * this chunk -- randomness is derived from the global index, so chunked keygen equals one-shot keygen.
 * Writes both parties' key buffers (fusefss_key_bytes() each, 256-byte aligned device memory). */
int fusefss_keygen(const fusefss_program *prog, const uint64_t *r_in_dev, const uint64_t *r_out_dev,
                   uint64_t seed, uint64_t first_elem, size_t count,
                   void *key0_dev, void *key1_dev, void *stream);

/* The same work split by key section, for per-kernel timing: parts = OR of FUSEFSS_GEN_CMP (the T bit-DCF keys),
 * FUSEFSS_GEN_LUT (the M-1 vector-DCF keys) and FUSEFSS_GEN_SHARES (c_b, masks, kappa, Beaver/AND/B2A material).
 * Calling the three parts in any order writes exactly what fusefss_keygen writes. */
enum { FUSEFSS_GEN_CMP = 1, FUSEFSS_GEN_LUT = 2, FUSEFSS_GEN_SHARES = 4 };
int fusefss_keygen_parts(const fusefss_program *prog, const uint64_t *r_in_dev, const uint64_t *r_out_dev,
                         uint64_t seed, uint64_t first_elem, size_t count,
                         void *key0_dev, void *key1_dev, int parts, void *stream);

/* ---- a5: packed comparison (section 3.6, Def I.1) --------------------------------
 * bits_out_dev[count]: bit t = this party's XOR share of I[view_{k_t,c_t}(xhat) < theta_t]. */
int fusefss_eval_cmp(int party, const fusefss_program *prog, const void *key_dev, const uint64_t *xhat_dev,
                     size_t count, uint64_t *bits_out_dev, void *stream);

/* ---- a6: vector interval lookup (section 3.6, Def I.2) ---------------------------
 * coeff_out_dev[p][count]: this party's additive share of the active interval's payload v_{i*} in R^p. */
int fusefss_eval_lut(int party, const fusefss_program *prog, const void *key_dev, const uint64_t *xhat_dev,
                     size_t count, uint64_t *coeff_out_dev, void *stream);

/* ---- a5 + a6 in one call -------------------------------------------------------------------------
 * Writes both outputs of the two FSS calls.  For variant 1 (single-key shared-prefix construction, DESIGN 9) both
 * come from ONE walk of the element's key at the public points xhat + delta_j, with the tree prefix shared by
 * nearby points; for variant 0 it is eval_cmp followed by eval_lut.  bits_out_dev may be NULL iff T = 0,
 * coeff_out_dev iff m = 1.  (eval_cmp / eval_lut remain valid for variant 1 and each walk only the points they need.) */
int fusefss_eval_fused(int party, const fusefss_program *prog, const void *key_dev, const uint64_t *xhat_dev,
                       size_t count, uint64_t *bits_out_dev, uint64_t *coeff_out_dev, void *stream);
/* The same for BOTH parties (one GPU runs both, north_star): for variant 1 a single launch walks both parties' keys
 * (half the launches, twice the parallelism for small tensors); otherwise two fusefss_eval_fused calls.  Outputs equal
 * the per-party calls bit for bit. */
int fusefss_eval_fused_both(const fusefss_program *prog, const void *key0_dev, const void *key1_dev,
                            const uint64_t *xhat_dev, size_t count, uint64_t *bits0_dev, uint64_t *bits1_dev,
                            uint64_t *coeff0_dev, uint64_t *coeff1_dev, void *stream);

/* ---- a7: post-processing (online steps 4-6; Horner P:895; DESIGN 4.6) ---------
 * One call per party per round.  msg_in_dev = the OTHER party's message buffer, msg_out_dev = this party's;
 * both cover all rounds (sum over q of fusefss_post_msg_bytes(q)).  round q in [0, rounds) writes this party's
 * openings of round q into msg_out_dev (replaying rounds < q from both buffers); round == rounds writes
 * y_out_dev[n_out_a][count] (shares of y, or of yhat = y + r_out when mask_output) and z_out_dev[count]
 * (bit j = XOR share of output bit j).  bits_dev / coeff_dev may be NULL when the respective call is omitted. */
int fusefss_post(int party, const fusefss_program *prog, const void *key_dev, const uint64_t *xhat_dev,
                 const uint64_t *bits_dev, const uint64_t *coeff_dev, size_t count, int round,
                 const void *msg_in_dev, void *msg_out_dev, uint64_t *y_out_dev, uint64_t *z_out_dev,
                 void *stream);
int fusefss_post_rounds(const fusefss_program *prog);
size_t fusefss_post_msg_bytes(const fusefss_program *prog, size_t count, int round);
/* algorithmic online bits per element per party: n (xhat) + n per opened ring element (2 per Beaver product, 1 per x-product,
 * 1 per interactive A2B) + 2 M_B + #B2A (+ n n_out_a if masked) */
size_t fusefss_online_bits(const fusefss_program *prog);
/* Both parties, all rounds, one launch; outputs equal the per-round API bit for bit. */
int fusefss_post_fused(const fusefss_program *prog, const void *key0_dev, const void *key1_dev,
                       const uint64_t *xhat_dev, const uint64_t *bits0_dev, const uint64_t *bits1_dev,
                       const uint64_t *coeff0_dev, const uint64_t *coeff1_dev, size_t count,
                       uint64_t *y0_dev, uint64_t *y1_dev, uint64_t *z0_dev, uint64_t *z1_dev, void *stream);

/* ---- a7 without any device allocation ----------------------------------------------------------------------
 * fusefss_post_fused_noalloc does exactly what fusefss_post_fused does (same arguments, same outputs bit for bit) but never
 * calls cudaMalloc / cudaFree or any routine that allocates device memory.
 *
 * Who needs it.  fusefss_post_fused keeps the lowered post-processing program (the instruction table its kernel interprets)
 * in a small device buffer that it cudaMalloc's the first time a program is used on a device.  Some hosts of this library
 * cannot afford or are not allowed that call:
 *   - an inference server whose tensor allocator has already reserved practically all of HBM for weights and caches, so a raw
 *     cudaMalloc from a third-party library fails with out-of-memory (or is forbidden by the server's memory accounting);
 *   - an online MPC loop with a latency budget: cudaMalloc synchronises the whole device, so a first-use allocation in the
 *     middle of a layer stalls every other stream of the process;
 *   - a party process confined to a fixed device-memory quota (MPS memory limit, container policy) sized in advance.
 * For those callers the instruction table lives in a fixed array that is part of the library image itself
 * (`static __device__`, FUSEFSS_NOALLOC_MAX_INS * 24 bytes = 48 KB): every GPU that loads libfusefss holds that array from
 * module load until the process exits, whether or not this function is ever called.
 *
 * Limit.  A program whose lowered post-processing code is longer than FUSEFSS_NOALLOC_MAX_INS instructions is rejected with
 * FUSEFSS_E_STATIC (every gate of the paper's benchmark suite lowers to well under 100).  That check needs no GPU and comes
 * before the count check, so `fusefss_post_fused_noalloc(prog, k0, k1, xhat, ..., count = 0, ...)` answers at start-up:
 * FUSEFSS_E_STATIC = does not fit, FUSEFSS_E_COUNT = fits.
 *
 * Set-up.  The first call on each device looks up the device address of the array (cudaGetSymbolAddress, with that device
 * current) and, like every entry point, uploads the PRG constants once (a synchronous cudaMemcpyToSymbol).  Make that first
 * call during start-up, before any stream capture begins on that device.
 *
 * Sharing.  There is ONE array per device, shared by every call, every program and every stream.  Each call copies its
 * program's instructions into the front of the array on `stream` (a few hundred bytes to a few KB, ordered before its kernel)
 * and whatever the previous call left behind stays there; nothing in the array has to start at zero, because the kernel reads
 * exactly the n_ins entries this call wrote.  Two calls whose GPU work can overlap -- different streams, or different host
 * threads on different streams -- race on the array and may interpret each other's program: serialise them (same stream, or an
 * event between them).  Calls on one stream are safe back to back.
 * Apart from that table the function uses no memory beyond the caller's inputs and outputs.  For the paper's Protocol-3
 * construction (variant bit 0 clear) fusefss_eval_cmp / _lut / _fused / _fused_both never allocate either, so the whole online
 * phase of a gate can run allocation-free. */
#define FUSEFSS_NOALLOC_MAX_INS 2048
int fusefss_post_fused_noalloc(const fusefss_program *prog, const void *key0_dev, const void *key1_dev,
                               const uint64_t *xhat_dev, const uint64_t *bits0_dev, const uint64_t *bits1_dev,
                               const uint64_t *coeff0_dev, const uint64_t *coeff1_dev, size_t count,
                               uint64_t *y0_dev, uint64_t *y1_dev, uint64_t *z0_dev, uint64_t *z1_dev, void *stream);

/* ---- vector-block glue (App. G: blocks = linear ops on shares + compiled scalar gates) ----------
 * fusefss_share_open: Protocol 1 for the input of gate `prog`: xhat = (x_0 + [r_in]_0) + (x_1 + [r_in]_1)
 *   + public_offset; the [r_in] shares are read from the two key buffers generated for these `count` elements (n/8 bytes
 *   per party).  public_offset = 2^{n-1} feeds the signed-truncation gate (workloads.specs.ars), 0 otherwise.
 * fusefss_open_output: online step 6 for a gate compiled with mask_output: yhat = y0 + y1 + public_offset, where y_b
 *   are the parties' shares of y + r_out written by fusefss_post / _post_fused (n/8 bytes per party).  When the NEXT gate is keyed
 *   with r_in = this gate's r_out, yhat is that gate's xhat: no second mask and no separate fusefss_share_open pass.
 * fusefss_sub_bcast: out[i] = x[i] - mu[i / cols] mod 2^n, local on additive shares.
 * fusefss_row_sum: out[r] = sum_c in[r*cols + c] mod 2^n, local on additive shares.
 * fusefss_mul_keygen / fusefss_mul_fused: element-wise Beaver products z = x * y (formulas DESIGN 4.6) with y
 *   broadcast over `cols` consecutive elements (cols = 1: plain element-wise; y has count/cols entries); the dealer's
 *   triples (fusefss_mul_triple_bytes(count) per party) come from R(e, 0xA000..0xA002); both parties in one launch,
 *   2n/8 online bytes per party per product. */
int fusefss_share_open(const fusefss_program *prog, const void *key0_dev, const void *key1_dev, const uint64_t *x0_dev,
                       const uint64_t *x1_dev, size_t count, uint64_t public_offset, uint64_t *xhat_out_dev, void *stream);
int fusefss_open_output(uint32_t n_bits, const uint64_t *y0_dev, const uint64_t *y1_dev, size_t count, uint64_t public_offset,
                        uint64_t *yhat_out_dev, void *stream);
int fusefss_sub_bcast(uint32_t n_bits, const uint64_t *x_dev, const uint64_t *mu_dev, size_t count, size_t cols,
                      uint64_t *out_dev, void *stream);
int fusefss_row_sum(uint32_t n_bits, const uint64_t *in_dev, size_t rows, size_t cols, uint64_t *out_dev, void *stream);
size_t fusefss_mul_triple_bytes(size_t count);
int fusefss_mul_keygen(uint32_t n_bits, uint64_t seed, uint64_t first_elem, size_t count, void *t0_dev, void *t1_dev, void *stream);
int fusefss_mul_fused(uint32_t n_bits, const uint64_t *x0_dev, const uint64_t *x1_dev, const uint64_t *y0_dev,
                      const uint64_t *y1_dev, const void *t0_dev, const void *t1_dev, size_t count, size_t cols,
                      uint64_t *z0_dev, uint64_t *z1_dev, void *stream);

/* ---- end-to-end convenience: HOST buffers in, HOST buffers out (bench.py's e2e leg) ---------------
 * Runs keygen + both parties' evaluation (one launch) + post_fused in chunks of `chunk` elements on `stream`, using the caller's
 * device workspace; r_in / r_out / xhat are copied to the device and y0, y1 [n_out_a][count], z0, z1 [count] back on an internal
 * copy stream, double-buffered, so the copies of chunk i+1 (in) and i-1 (out) overlap the kernels of chunk i (pin the host
 * buffers for that).  Returns after everything has completed.  workspace_dev must hold fusefss_gate_workspace_bytes(prog, chunk)
 * bytes; workspace_bytes is what the caller allocated (FUSEFSS_E_WORKSPACE if it is too small).  Calls on one device are serialised
 * (they share that device's copy stream and events); calls on different devices of one process run concurrently.  On an error return
 * both streams have been drained first: no copy into the caller's host buffers is still in flight. */
size_t fusefss_gate_workspace_bytes(const fusefss_program *prog, size_t chunk);
int fusefss_gate_host(const fusefss_program *prog, const uint64_t *r_in, const uint64_t *r_out,
                      const uint64_t *xhat, uint64_t seed, size_t count, size_t chunk, void *workspace_dev,
                      size_t workspace_bytes, uint64_t *y0, uint64_t *y1, uint64_t *z0, uint64_t *z1, void *stream);

/* ---- algorithmic work per element (for the roofline; DESIGN 5.3, 9) ---------------------------------
 * AES-128 blocks and T-table lookups of one party's evaluation (cmp part / lut part; for variant 1 "lut" = the fused
 * walk of the n-bit tree, "cmp" = the narrower bit trees) and of the dealer's keygen (both bundles), plus the key
 * bytes one party's evaluation reads. */
typedef struct {
    uint64_t eval_cmp_aes, eval_cmp_lookups, eval_lut_aes, eval_lut_lookups;
    uint64_t gen_cmp_aes, gen_cmp_lookups, gen_lut_aes, gen_lut_lookups;
    uint64_t eval_cmp_key_bytes, eval_lut_key_bytes;
} fusefss_cost_t;
int fusefss_cost(const fusefss_program *prog, fusefss_cost_t *out);

/* ---- diagnostics ---------------------------------------------------------------------------------- */
const char *fusefss_strerror(int code);
const char *fusefss_last_cuda_error(void);
/* Test / tuning knobs (process-wide, not part of the method): "force_g" = v >= 1 forces the number of warps the trees / points of an
 * element are dealt to (0 = automatic); "eval_threads" = CTA size of the large evaluation launches (default 1024); "small_kernels"
 * = 0 disables the 256-thread instantiations used for small launches; "sp_np" = points the single-key evaluation walks in lock-step per
 * warp (0 = automatic); "gen_quad" = 0 disables the four-lanes-per-element dealer kernel used for small launches; "coop" = 0: launches that accumulate with
 * atomics clear their outputs with cudaMemsetAsync and launch normally instead of zeroing in-kernel behind a cooperative-launch grid barrier (the
 * library takes that road by itself when the context refuses the cooperative launch); "sp_split" = 0 / 1 / 2: the lane-split
 * single-key evaluation kernel never / for tiny launches (default) / for every small launch.  Unknown knob: FUSEFSS_E_DEBUG. */
int fusefss_debug_set(const char *knob, long value);
/* number of kernel launches this library has issued since load (bench.py's gpu_launches) */
uint64_t fusefss_launch_count(void);
/* PRG micro-kernel for the roofline denominator: each thread chains `iters` fixed-key AES-128 blocks starting
 * from its index and writes the last block to out_dev[threads*16 bytes]; blocks = threads*iters. */
int fusefss_aes_probe(size_t threads, int iters, void *out_dev, void *stream);
/* Latency probe for the small-tensor floor: ONE warp chains `trips` dependent trips, each expanding the lane's seed into blocks_per_trip
 * (1..5) AES blocks that share their round-1 lookups -- the PRG work of one level of a tree with that many blocks per node, 32 elements in
 * lock-step, with no key loads and no tree logic.  One 256-thread CTA (launch + table fill cost what a small evaluation launch pays).
 * out_dev holds 32 * 16 bytes.  FUSEFSS_E_COUNT for trips <= 0 or blocks_per_trip outside 1..5. */
int fusefss_aes_chain_probe(int blocks_per_trip, int trips, void *out_dev, void *stream);
/* Pipe micro-probes for the roofline denominators: kind 0 = LOP3 issue (8 independent chains per thread), kind 1 =
 * conflict-free LDS.32 wavefronts (8 dependent-lookup chains per thread through the bank-replicated table).  One CTA of
 * 1024 threads per SM; out_dev holds SMs*1024 uint32.  Operations executed = SMs * 1024 * 8 * iters (lane-ops). */
int fusefss_pipe_probe(int kind, int iters, void *out_dev, void *stream);
/* A bitsliced AES-128 core (32 blocks per thread as 128 bit-planes, composite-field S-box circuit), built only to TIME it against the
 * T-table core (DESIGN 5.2).  _kat: in_dev / out_dev = 32 blocks of 16 bytes (device), one encryption with key[16] (HOST).
 * _probe: each of `threads` threads chains `iters` encryptions of its 32 blocks; out_dev holds threads*16 bytes; blocks =
 * threads * 32 * iters. */
int fusefss_bitslice_kat(const uint8_t *key, const void *in_dev, void *out_dev, void *stream);
int fusefss_bitslice_probe(const uint8_t *key, size_t threads, int iters, void *out_dev, void *stream);
/* single-block AES-128 (FIPS-197) through the device PRG core, for the known-answer test: key[16], in[16] HOST,
 * out_dev[16] device */
int fusefss_aes_kat(const uint8_t *key, const uint8_t *in, void *out_dev, void *stream);

#ifdef __cplusplus
}
#endif
#endif /* FUSEFSS_H */
