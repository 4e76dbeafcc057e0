// omerf_mlp.cuh — the deferred MLP G of Eq. 4 on tensor cores, shared by the march kernel's retire
// phase (omerf_render.cu) and the batched smoothness workload (omerf_smooth.cu).  Internal to the CUDA path.
#pragma once
#include "omerf_device.cuh"

namespace {

__device__ __forceinline__ float sigmoid_fast(float x) { return __fdividef(1.0f, 1.0f + __expf(-x)); }

// ---------------------------------------------------------------------------------- S8: deferred MLP (Eq. 4)
// Warp-cooperative: the 34 -> 16 -> 16 -> 3 network of 16 rays at a time as m16n8k8 tensor-core tiles.
// tf32 operands are split hi + lo (3 mma per tile product), so the result keeps fp32-level accuracy; hidden
// activations stay in registers (the C fragment of one layer is the A fragment of the next, see mlp_pack_kernel).

// x = hi + lo with hi = x truncated to tf32 (10 explicit mantissa bits) and lo = x - hi exactly; the tensor core
// reads only the tf32 part of lo, which leaves a relative error of about 2^-21 in the product sum
__device__ __forceinline__ void split_tf32(float x, uint32_t &hi, uint32_t &lo)
{
    hi = __float_as_uint(x) & 0xffffe000u;
    lo = __float_as_uint(x - __uint_as_float(hi));
}

__device__ __forceinline__ void mma_tf32(float c[4], const uint32_t a[4], float b0, float b1)
{
    asm volatile("mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                 : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
                 : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(__float_as_uint(b0)), "r"(__float_as_uint(b1)));
}

// c += A * B for one k-step/n-tile, A given as fp32 values (split here), B from the packed table
__device__ __forceinline__ void mma_x3(float c[4], const uint32_t ahi[4], const uint32_t alo[4], const float2 *__restrict__ tab,
                                       int tile, int lane)
{
    const float2 bhi = __ldg(tab + (tile * 2 + 0) * 32 + lane), blo = __ldg(tab + (tile * 2 + 1) * 32 + lane);
    mma_tf32(c, alo, bhi.x, bhi.y);
    mma_tf32(c, ahi, blo.x, blo.y);
    mma_tf32(c, ahi, bhi.x, bhi.y);
}

// Column order of the layer-1 input matrix (K = 34, padded to 40).  An m16n8k8 A fragment gives lane (g, t) the columns
// 8s + t and 8s + t + 4 of k-step s, i.e. ten values v[2s], v[2s + 1] per row.  The 34 inputs of Eq. 4 (R13:
// sum w c^d (3), sum w f (4), d (3), sin/cos(2^j d), j = 0..3) are laid out so that one lane can produce its ten values
// from ONE direction component (no staging through shared memory):
//   t = 0,1,2 (component c = t):  v = [d_c, sin d_c, cos d_c, sin 2d_c, cos 2d_c, sin 4d_c, cos 4d_c, sin 8d_c, cos 8d_c, acc_t]
//   t = 3:                        v = [acc_3, acc_4, acc_5, acc_6, -, -, -, -, -, -]   (- : weight 0, any finite value)
// mlp_pack_kernel (omerf_build.cu) permutes the columns of W0 with mlp_orig_of_col (omerf_device.cuh), so the network is
// unchanged.
// d, then sin/cos(2^j d), j = 0..3, of one direction component: v[0..8]
// FAST: sin/cos of d through the MUFU intrinsics (absolute error 2^-21.4 on [-pi, pi], about 3e-6 after the three angle
// doublings, i.e. <= 4e-6 on an output colour): used by the renderer (budget 2e-3), not by the smoothness term, which
// differences G.
template <bool FAST>
__device__ __forceinline__ void mlp_encode_component(float d, float v[9])
{
    float s, co;
    if (FAST) __sincosf(d, &s, &co);
    else sincosf(d, &s, &co); // |d| <= 1: no range-reduction slow path
    v[0] = d;
#pragma unroll
    for (int j = 0; j < 4; j++) {
        v[1 + 2 * j] = s;
        v[2 + 2 * j] = co;
        const float s2 = 2.0f * s * co, c2 = 1.0f - 2.0f * s * s; // double angle: sin/cos(2^(j+1) d)
        s = s2;
        co = c2;
    }
}

// Evaluates G for 16 rows given as register fragments: v0 = this lane's ten layer-1 values of row g, v1 = of row g + 8
// (column order above).  Returns this lane's share of the output C fragment: out[0], out[1] = row g cols 2t, 2t+1;
// out[2], out[3] = row g+8 (pre-sigmoid; cols >= 3 unused).
__device__ __forceinline__ void mlp_tiles(const float2 *__restrict__ tab, const float v0[10], const float v1[10], int lane, float out[4])
{
    float c1[2][4], c2[2][4];
#pragma unroll
    for (int q = 0; q < 2; q++) {
        const float2 bq = __ldg(tab + OMERF_MLP_BIAS_OFF + q * 32 + lane), bq2 = __ldg(tab + OMERF_MLP_BIAS_OFF + (2 + q) * 32 + lane);
        c1[q][0] = c1[q][2] = bq.x;
        c1[q][1] = c1[q][3] = bq.y;
        c2[q][0] = c2[q][2] = bq2.x;
        c2[q][1] = c2[q][3] = bq2.y;
    }
    // layer 1: K = 34 (padded to 40), N = 16
#pragma unroll
    for (int s = 0; s < 5; s++) {
        uint32_t ahi[4], alo[4];
        split_tf32(v0[2 * s], ahi[0], alo[0]);
        split_tf32(v1[2 * s], ahi[1], alo[1]);
        split_tf32(v0[2 * s + 1], ahi[2], alo[2]);
        split_tf32(v1[2 * s + 1], ahi[3], alo[3]);
#pragma unroll
        for (int q = 0; q < 2; q++) mma_x3(c1[q], ahi, alo, tab, s * 2 + q, lane);
    }
    // layer 2: K = 16, N = 16; A fragment of k-step s = relu(C fragment of n-tile s)
#pragma unroll
    for (int s = 0; s < 2; s++) {
        uint32_t ahi[4], alo[4];
        split_tf32(fmaxf(c1[s][0], 0.0f), ahi[0], alo[0]);
        split_tf32(fmaxf(c1[s][2], 0.0f), ahi[1], alo[1]);
        split_tf32(fmaxf(c1[s][1], 0.0f), ahi[2], alo[2]);
        split_tf32(fmaxf(c1[s][3], 0.0f), ahi[3], alo[3]);
#pragma unroll
        for (int q = 0; q < 2; q++) mma_x3(c2[q], ahi, alo, tab, 10 + s * 2 + q, lane);
    }
    // layer 3: K = 16, N = 3 (padded to 8)
    const float2 b3 = __ldg(tab + OMERF_MLP_BIAS_OFF + 4 * 32 + lane);
    out[0] = out[2] = b3.x;
    out[1] = out[3] = b3.y;
#pragma unroll
    for (int s = 0; s < 2; s++) {
        uint32_t ahi[4], alo[4];
        split_tf32(fmaxf(c2[s][0], 0.0f), ahi[0], alo[0]);
        split_tf32(fmaxf(c2[s][2], 0.0f), ahi[1], alo[1]);
        split_tf32(fmaxf(c2[s][1], 0.0f), ahi[2], alo[2]);
        split_tf32(fmaxf(c2[s][3], 0.0f), ahi[3], alo[3]);
        mma_x3(out, ahi, alo, tab, 14 + s, lane);
    }
}

} // namespace
