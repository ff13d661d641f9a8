// blocks.cuh -- linear glue for vector blocks composed from compiled gates (App. G,
// softmax = nExp -> sum -> Recip -> Beaver product; the max reduction is not compiled).
// Everything here is bandwidth-trivial: masked opening of a gate input (Protocol 1), row sums of
// additive shares, and element-wise Beaver products with an optional per-row broadcast operand.
#pragma once
#include <cstdint>

#include "aes.cuh"
#include "keygen.cuh"

namespace fsk {

// Protocol 1: xhat = (x_0 + [r_in]_0) + (x_1 + [r_in]_1) mod 2^n; each party sends one ring element.
struct OpenArgs { const uint64_t *x0, *x1; const uint8_t *key0, *key1; size_t rin_off, count; uint64_t mask, offset; uint64_t *xhat; };
__global__ void k_share_open(const OpenArgs a) {
    const size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= a.count) return;
    const uint64_t r0 = reinterpret_cast<const uint64_t *>(a.key0 + a.rin_off)[e], r1 = reinterpret_cast<const uint64_t *>(a.key1 + a.rin_off)[e];
    a.xhat[e] = (a.x0[e] + r0 + a.x1[e] + r1 + a.offset) & a.mask;      // offset: public constant added to the gate input
}

// Online step 6: opening of a masked output yhat = y + r_out from the two parties' shares of it (each sends one
// ring element).  With r_in(next gate) = r_out(this gate) the public yhat IS the next gate's xhat.
struct OpenOutArgs { const uint64_t *y0, *y1; size_t count; uint64_t mask, offset; uint64_t *yhat; };
__global__ void k_open_output(const OpenOutArgs a) {
    const size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e < a.count) a.yhat[e] = (a.y0[e] + a.y1[e] + a.offset) & a.mask;
}

// out[r] = sum_c in[r*cols + c] mod 2^n (local on additive shares): one warp per row
struct RowSumArgs { const uint64_t *in; uint64_t *out; size_t rows, cols; uint64_t mask; };
__global__ void k_row_sum(const RowSumArgs a) {
    const size_t row = ((size_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    if (row >= a.rows) return;
    const int lane = threadIdx.x & 31;
    uint64_t acc = 0;
    for (size_t c = lane; c < a.cols; c += 32) acc += a.in[row * a.cols + c];
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, off);
    if (lane == 0) a.out[row] = acc & a.mask;
}

// out[i] = x[i] - mu[i / cols] mod 2^n (local on additive shares): centring by a per-row value
struct SubBcastArgs { const uint64_t *x, *mu; uint64_t *out; size_t count, cols; uint64_t mask; };
__global__ void k_sub_bcast(const SubBcastArgs a) {
    const size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e < a.count) a.out[e] = (a.x[e] - a.mu[e / a.cols]) & a.mask;
}

// Beaver triples for `count` products: per party [a][b][c] arrays of s8 bytes each; randomness R(e, 0xA000..0xA002)
enum : uint64_t { SLOT_MUL_AB = 0xA000, SLOT_MUL_AB0 = 0xA001, SLOT_MUL_C0 = 0xA002 };
struct MulGenArgs { uint8_t *t0, *t1; size_t count, s8; uint64_t first_elem, mask; RoundKeys rk; };
__global__ void __launch_bounds__(kGenThreads, 1) k_mul_gen(const __grid_constant__ MulGenArgs a) {
    extern __shared__ uint32_t sT[];
    const uint32_t tl = aes_fill_tables(sT);
    for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < a.count; e += (size_t)gridDim.x * blockDim.x) {
        uint64_t lo, hi;
        dealer_rand(tl, a.rk, a.first_elem + e, SLOT_MUL_AB, lo, hi);
        const uint64_t ta = lo & a.mask, tb = hi & a.mask, tc = (ta * tb) & a.mask;
        dealer_rand(tl, a.rk, a.first_elem + e, SLOT_MUL_AB0, lo, hi);
        const uint64_t a0 = lo & a.mask, b0 = hi & a.mask;
        dealer_rand(tl, a.rk, a.first_elem + e, SLOT_MUL_C0, lo, hi);
        const uint64_t c0 = lo & a.mask;
        uint64_t *p0 = reinterpret_cast<uint64_t *>(a.t0), *p1 = reinterpret_cast<uint64_t *>(a.t1);
        const size_t w = a.s8 / 8;
        p0[e] = a0; p0[w + e] = b0; p0[2 * w + e] = c0;
        p1[e] = (ta - a0) & a.mask; p1[w + e] = (tb - b0) & a.mask; p1[2 * w + e] = (tc - c0) & a.mask;
    }
}

// z = x * y element-wise, y broadcast over `cols` consecutive elements (cols = 1: plain element-wise); both parties in
// one pass: open e = x - a, f = y - b;  [z]_b = [b=0] e f + e [b]_b + f [a]_b + [c]_b   (DESIGN 4.6)
struct MulArgs { const uint64_t *x0, *x1, *y0, *y1; const uint8_t *t0, *t1; uint64_t *z0, *z1; size_t count, cols, s8; uint64_t mask; };
__global__ void k_mul_fused(const MulArgs a) {
    const size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= a.count) return;
    const size_t w = a.s8 / 8, yi = e / a.cols;
    const uint64_t *p0 = reinterpret_cast<const uint64_t *>(a.t0), *p1 = reinterpret_cast<const uint64_t *>(a.t1);
    const uint64_t a0 = p0[e], b0 = p0[w + e], c0 = p0[2 * w + e], a1 = p1[e], b1 = p1[w + e], c1 = p1[2 * w + e];
    const uint64_t E = ((a.x0[e] - a0) + (a.x1[e] - a1)) & a.mask, Fv = ((a.y0[yi] - b0) + (a.y1[yi] - b1)) & a.mask;
    a.z0[e] = (E * Fv + E * b0 + Fv * a0 + c0) & a.mask;
    a.z1[e] = (E * b1 + Fv * a1 + c1) & a.mask;
}

}  // namespace fsk
