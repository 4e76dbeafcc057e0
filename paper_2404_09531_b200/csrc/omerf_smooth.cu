// omerf_smooth.cu — view-direction smoothness term (Eq. 9-10) as a batched
// workload of the deferred MLP G (Eq. 4):
//     l(d) = sum_s S(d, s) || G(F, s) - G(F, d) ||^2,   s = d + delta,   S = cosine similarity.
// One warp per viewing direction; its 1 + S evaluations of G run as 16-row tensor-core tiles (omerf_mlp.cuh), row 0 of
// the first tile being G(F, d).  Lane (g, t) builds its layer-1 A fragment of rows g and g + 8 in registers from ONE
// component of s (column order of omerf_mlp.cuh): nothing is staged through shared memory.  The perturbed direction goes
// into the encoding as it is (R25).
#include "omerf_device.cuh"
#include "omerf_mlp.cuh"

namespace {

constexpr int SMOOTH_WARPS = 4;
constexpr int SMOOTH_MIN_BLOCKS = 7; // 72 registers, 28 warps per SM: 0.924 ms; 6 blocks 0.970, 8 blocks (64 registers) 0.952, 4 blocks (121 registers) 1.13

struct SmoothDir {          // what a lane keeps of one direction
    float d[3];             // the direction
    float f9, f1, f2, f3;   // F[t] (t = 3: F[3]); F[4..6] for lanes t = 3
};

__device__ __forceinline__ void smooth_fetch(long long i, int t, const float *__restrict__ F, const float *__restrict__ dir, SmoothDir &q)
{
    q.d[0] = __ldg(dir + i * 3 + 0);
    q.d[1] = __ldg(dir + i * 3 + 1);
    q.d[2] = __ldg(dir + i * 3 + 2);
    q.f9 = __ldg(F + i * 7 + t);
    q.f1 = __ldg(F + i * 7 + 4);
    q.f2 = __ldg(F + i * 7 + 5);
    q.f3 = __ldg(F + i * 7 + 6);
}

// One tile of 16 rows j = 16 tile + (0..15) of direction i (row 0 = d itself): returns this lane's two rows' colours
// (sigmoid applied; c[0], c[1] = row g cols 2t, 2t+1; c[2], c[3] = row g + 8) and their weights S(d, s) (0 for row 0 and
// for rows past S).
__device__ __forceinline__ void smooth_tile(const float2 *__restrict__ tab, const SmoothDir &q, long long i, int S, int tile,
                                            const float *__restrict__ delta, int lane, float c[4], float w[2])
{
    const int g = lane >> 2, t = lane & 3, comp = min(t, 2);
    float v[2][10];
#pragma unroll
    for (int rr = 0; rr < 2; rr++) {
        const int j = tile * 16 + g + 8 * rr;
        float sx = q.d[0], sy = q.d[1], sz = q.d[2];
        w[rr] = 0.0f;
        if (j > 0 && j <= S) {
            const float *dl = delta + (i * S + (j - 1)) * 3;
            sx = __fadd_rn(sx, __ldg(dl + 0));
            sy = __fadd_rn(sy, __ldg(dl + 1));
            sz = __fadd_rn(sz, __ldg(dl + 2));
            const float dot = q.d[0] * sx + q.d[1] * sy + q.d[2] * sz;
            const float nn = (q.d[0] * q.d[0] + q.d[1] * q.d[1] + q.d[2] * q.d[2]) * (sx * sx + sy * sy + sz * sz);
            w[rr] = nn > 0.0f ? dot * rsqrtf(nn) : 0.0f;
        }
        mlp_encode_component<false>(comp == 0 ? sx : (comp == 1 ? sy : sz), v[rr]);
        v[rr][9] = q.f9;
        if (t == 3) {
            v[rr][0] = q.f9;
            v[rr][1] = q.f1;
            v[rr][2] = q.f2;
            v[rr][3] = q.f3;
        }
    }
    float o[4];
    mlp_tiles(tab, v[0], v[1], lane, o);
#pragma unroll
    for (int k = 0; k < 4; k++) c[k] = sigmoid_fast(o[k]);
}

// loss terms of this lane's two rows of a tile; lane (g, t): t = 0 holds colours 0,1 and t = 1 colour 2
__device__ __forceinline__ float smooth_terms(const float c[4], const float w[2], const float G0[3], long long i, int S, int tile,
                                              int lane, float *__restrict__ out_G)
{
    const int g = lane >> 2, t = lane & 3;
    float loss = 0.0f;
    if (t < 2) {
#pragma unroll
        for (int rr = 0; rr < 2; rr++) {
            const int j = tile * 16 + g + 8 * rr;
            if (j <= S) {
                if (t == 0) {
                    const float a = c[2 * rr] - G0[0], b = c[2 * rr + 1] - G0[1];
                    loss += w[rr] * (a * a + b * b);
                } else {
                    const float a = c[2 * rr] - G0[2];
                    loss += w[rr] * a * a;
                }
                if (out_G) {
                    float *og = out_G + (i * (S + 1) + j) * 3;
                    if (t == 0) {
                        og[0] = c[2 * rr];
                        og[1] = c[2 * rr + 1];
                    } else {
                        og[2] = c[2 * rr];
                    }
                }
            }
        }
    }
    return loss;
}

// G(F, d) = row 0 of tile 0: lane 0 holds colours 0,1, lane 1 colour 2
__device__ __forceinline__ void smooth_G0(const float c[4], float G0[3])
{
    const unsigned FULL = 0xffffffffu;
    G0[0] = __shfl_sync(FULL, c[0], 0);
    G0[1] = __shfl_sync(FULL, c[1], 0);
    G0[2] = __shfl_sync(FULL, c[0], 1);
}

__device__ __forceinline__ float warp_sum(float x)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
    return x;
}

__global__ void __launch_bounds__(32 * SMOOTH_WARPS, SMOOTH_MIN_BLOCKS)
omerf_smooth_kernel(const float2 *__restrict__ mlp_tab, long long n, int S, const float *__restrict__ F,
                    const float *__restrict__ dir, const float *__restrict__ delta, float *__restrict__ out_loss,
                    float *__restrict__ out_G)
{
    const int lane = threadIdx.x & 31, t = lane & 3;
    const long long warps = (long long)gridDim.x * SMOOTH_WARPS, w0 = (long long)blockIdx.x * SMOOTH_WARPS + (threadIdx.x >> 5);
    const int tiles = (S + 16) / 16;
    for (long long i = w0; i < n; i += warps) {
        SmoothDir q;
        smooth_fetch(i, t, F, dir, q);
        float G0[3] = {0.0f, 0.0f, 0.0f}, loss = 0.0f;
        for (int tile = 0; tile < tiles; tile++) {
            float c[4], w[2];
            smooth_tile(mlp_tab, q, i, S, tile, delta, lane, c, w);
            if (tile == 0) smooth_G0(c, G0);
            loss += smooth_terms(c, w, G0, i, S, tile, lane, out_G);
        }
        loss = warp_sum(loss);
        if (lane == 0) out_loss[i] = loss;
    }
}

} // namespace

int omerf_launch_smoothness(const omerf_scene *s, long long n, int S, const float *F, const float *dir, const float *delta,
                            float *out_loss, float *out_G, cudaStream_t st)
{
    if (n == 0) return OMERF_OK;
    int dev = 0, sms = 0;
    OMERF_CUDA(cudaGetDevice(&dev));
    OMERF_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    long long blocks = (n + SMOOTH_WARPS - 1) / SMOOTH_WARPS;
    int per_sm = 0;
    OMERF_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, omerf_smooth_kernel, 32 * SMOOTH_WARPS, 0));
    const long long cap = (long long)sms * (per_sm > 0 ? per_sm : 1); // persistent grid: one wave of resident CTAs
    if (blocks > cap) blocks = cap;
    omerf_smooth_kernel<<<(unsigned int)blocks, 32 * SMOOTH_WARPS, 0, st>>>(s->dev.mlp_tab, n, S, F, dir, delta, out_loss, out_G);
    OMERF_CUDA(cudaGetLastError());
    return OMERF_OK;
}
