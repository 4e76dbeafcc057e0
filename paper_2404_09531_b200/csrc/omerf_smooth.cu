// omerf_smooth.cu — view-direction smoothness term (Eq. 9-10) as a batched
// workload of the deferred MLP G (Eq. 4):
//     l(d) = sum_s S(d, s) || G(F, s) - G(F, d) ||^2,   s = d + delta,   S = cosine similarity.
// One warp per viewing direction; its 1 + S evaluations of G run as 16-row tensor-core tiles (omerf_mlp.cuh),
// two tiles per pass (lanes 0-15 stage one, lanes 16-31 the other).  Row 0 of the first tile is G(F, d).
// The perturbed direction goes into the encoding as it is (R25).
#include "omerf_device.cuh"
#include "omerf_mlp.cuh"

namespace {

#ifndef SMOOTH_WARPS
#define SMOOTH_WARPS 4
#endif

#ifndef SMOOTH_MIN_BLOCKS
#define SMOOTH_MIN_BLOCKS 5
#endif
__global__ void __launch_bounds__(32 * SMOOTH_WARPS, SMOOTH_MIN_BLOCKS)
omerf_smooth_kernel(const float2 *__restrict__ mlp_tab, long long n, int S, const float *__restrict__ F,
                    const float *__restrict__ dir, const float *__restrict__ delta, float *__restrict__ out_loss,
                    float *__restrict__ out_G)
{
    __shared__ float Xs[SMOOTH_WARPS][2][16 * OMERF_XS];
    __shared__ float Ws[SMOOTH_WARPS][2][16]; // S(d, s) of every staged row (0 for padding rows and for row 0)
    const unsigned FULL = 0xffffffffu;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int half = lane >> 4, row = lane & 15;
    const long long warps = (long long)gridDim.x * SMOOTH_WARPS;
    const int rows_total = S + 1, passes = (rows_total + 31) / 32;
    const int g = lane >> 2, t = lane & 3;

    // inputs of the first pass are fetched one direction ahead, so their DRAM latency overlaps the previous tiles
    struct In {
        float f7[7], dx, dy, dz, lx, ly, lz;
    };
    auto fetch = [&](long long i, In &q) {
        if (i >= n) return;
#pragma unroll
        for (int c = 0; c < 7; c++) q.f7[c] = __ldg(F + i * 7 + c);
        q.dx = __ldg(dir + i * 3 + 0);
        q.dy = __ldg(dir + i * 3 + 1);
        q.dz = __ldg(dir + i * 3 + 2);
        q.lx = q.ly = q.lz = 0.0f;
        if (lane > 0 && lane < rows_total) {
            const float *dl = delta + (i * S + (lane - 1)) * 3;
            q.lx = __ldg(dl + 0);
            q.ly = __ldg(dl + 1);
            q.lz = __ldg(dl + 2);
        }
    };
    In cur, nxt;
    fetch((long long)blockIdx.x * SMOOTH_WARPS + w, nxt);
    for (long long i = (long long)blockIdx.x * SMOOTH_WARPS + w; i < n; i += warps) {
        cur = nxt;
        fetch(i + warps, nxt);
        float f7[7];
#pragma unroll
        for (int c = 0; c < 7; c++) f7[c] = cur.f7[c];
        const float dx = cur.dx, dy = cur.dy, dz = cur.dz;
        float G0[3] = {0.f, 0.f, 0.f};
        float loss = 0.0f;
        for (int p = 0; p < passes; p++) {
            // ---- stage 32 rows: row j = 32 p + lane; j = 0 is the unperturbed direction
            const int j = p * 32 + lane;
            float in[40];
#pragma unroll
            for (int q = 0; q < 40; q++) in[q] = 0.0f;
            float cosv = 0.0f;
            if (j < rows_total) {
                float sx = dx, sy = dy, sz = dz;
                if (j > 0) {
                    float lx = cur.lx, ly = cur.ly, lz = cur.lz;
                    if (p > 0) {
                        const float *dl = delta + (i * S + (j - 1)) * 3;
                        lx = __ldg(dl + 0);
                        ly = __ldg(dl + 1);
                        lz = __ldg(dl + 2);
                    }
                    sx = __fadd_rn(dx, lx);
                    sy = __fadd_rn(dy, ly);
                    sz = __fadd_rn(dz, lz);
                    const float dot = dx * sx + dy * sy + dz * sz;
                    const float nn = (dx * dx + dy * dy + dz * dz) * (sx * sx + sy * sy + sz * sz);
                    cosv = nn > 0.0f ? dot * rsqrtf(nn) : 0.0f;
                }
                mlp_input<false>(f7, sx, sy, sz, in);
            }
            float4 *xr = reinterpret_cast<float4 *>(Xs[w][half] + row * OMERF_XS);
#pragma unroll
            for (int q = 0; q < 10; q++) xr[q] = make_float4(in[4 * q], in[4 * q + 1], in[4 * q + 2], in[4 * q + 3]);
            Ws[w][half][row] = cosv;
            __syncwarp();
            // ---- two tiles of 16 rows through G
#pragma unroll 1
            for (int tile = 0; tile < 2; tile++) {
                if (p * 32 + tile * 16 >= rows_total) break;
                float o[4];
                mlp_half(mlp_tab, Xs[w][tile], lane, o);
                // lane (g, t): t = 0 holds colours 0,1 and t = 1 colour 2 of rows g and g + 8 of this tile
                float c[4];
#pragma unroll
                for (int q = 0; q < 4; q++) c[q] = sigmoid_fast(o[q]);
                if (p == 0 && tile == 0) { // row 0 lives in lanes g = 0 (lane 0: colours 0,1; lane 1: colour 2)
                    G0[0] = __shfl_sync(FULL, c[0], 0);
                    G0[1] = __shfl_sync(FULL, c[1], 0);
                    G0[2] = __shfl_sync(FULL, c[0], 1);
                }
#pragma unroll
                for (int rr = 0; rr < 2; rr++) {
                    const int r16 = g + 8 * rr;
                    const int jj = p * 32 + tile * 16 + r16;
                    if (jj < rows_total && t < 2) {
                        const float wgt = Ws[w][tile][r16];
                        if (t == 0) {
                            const float a = c[2 * rr] - G0[0], b = c[2 * rr + 1] - G0[1];
                            loss += wgt * (a * a + b * b);
                        } else {
                            const float a = c[2 * rr] - G0[2];
                            loss += wgt * a * a;
                        }
                        if (out_G) {
                            float *og = out_G + (i * rows_total + jj) * 3;
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
            __syncwarp();
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) loss += __shfl_xor_sync(FULL, loss, o);
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
