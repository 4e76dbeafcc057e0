// omerf_build.cu — one-time scene derivations on the device.
//   S1  min/max pyramid of the occupancy plane: "2D max pooling to obtain multiple low-resolution
//       occupancy planes"; we min-pool z_min and max-pool z_max (R16).
//   S10 config-4 comparator: binary occupancy grid derived from the slab (voxel set iff it intersects
//       [z_min, z_max] of an overlapping cell, R18) and its OR-reduced mip chain — the
//       "multi-resolution binary grid" PAPER.md:188 says the occupancy plane replaces.
#include <string.h>

#include "omerf_device.cuh"

// ------------------------------------------------------------------------------------------ S0: gather layout
// Every feature array is stored as ENTRIES of two texels adjacent along one of its axes (y for V, the second axis for the
// planes):  dst[e] = pair_entry(src[e], src[e + stride]) (the texel itself again at the last index of that axis),
// 8 + 8 = 16 bytes with the two texels' bytes interleaved channel by channel (omerf_device.cuh: pair_entry).
// The two taps a bilinear / trilinear footprint takes along that axis arrive with ONE 16-byte load, already in the operand
// order of the 16-bit x 8-bit dot products that filter them: 10 gathers per sample instead of 20, no byte shuffles, for
// twice the memory (PAPER.md:186 stores the features as textures; SURVEY 8(a) S0 "re-lay out for gathers").  The repeated
// texel reproduces clamp-to-edge addressing (R10) at the last index; the first index needs none (omerf_render.cu: axis_tap).
__global__ void pair_layout_kernel(const uint2 *__restrict__ src, uint4 *__restrict__ dst, unsigned long long total, int n,
                                   unsigned long long stride)
{
    for (unsigned long long e = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; e < total;
         e += (unsigned long long)gridDim.x * blockDim.x) {
        const int j = (int)((e / stride) % (unsigned long long)n); // coordinate along the paired axis
        dst[e] = pair_entry(src[e], src[j + 1 < n ? e + stride : e]);
    }
}

// `total` texels; the paired axis has n texels and element stride `stride` (1: the fastest axis)
int omerf_launch_pair_layout(const void *d_src, void *d_dst, unsigned long long total, int n, unsigned long long stride, cudaStream_t st)
{
    if (total == 0 || n <= 0) return OMERF_OK;
    const unsigned int blocks = (unsigned int)((total + 255) / 256 < (1u << 20) ? (total + 255) / 256 : (1u << 20));
    pair_layout_kernel<<<blocks, 256, 0, st>>>((const uint2 *)d_src, (uint4 *)d_dst, total, n, stride);
    OMERF_CUDA(cudaGetLastError());
    return OMERF_OK;
}

// ------------------------------------------------------------------------------------------ low-z triplane bake
// "For the 2D triplane, we employ a texture map with high resolution in the xy direction and low resolution
// in the z direction, according to the upper and lower bounds of the occupancy plane."  DESIGN.md R27: the xz and yz
// planes keep the band of z rows a bilinear lookup can touch for z in [min z_min, max z_max] over the non-empty columns
// of P_o (clipped to the box, widened by 1/64 texel).  Step 1: the two bounds (ordered-integer keys, atomics);
// step 2: the band of each plane, in double with one rounding per operation.
__device__ __forceinline__ unsigned int lowz_key(float f)
{
    const unsigned int b = __float_as_uint(f);
    return (b & 0x80000000u) ? ~b : (b | 0x80000000u); // monotone in f
}

__device__ __forceinline__ float lowz_unkey(unsigned int k) { return __uint_as_float((k & 0x80000000u) ? (k & 0x7fffffffu) : ~k); }

__global__ void lowz_bounds_kernel(const float *__restrict__ lo, const float *__restrict__ up, int n, unsigned int *__restrict__ keys)
{
    unsigned int kmin = 0xffffffffu, kmax = 0u;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const float a = lo[i], b = up[i];
        if (a <= b) { // non-empty column (R17)
            kmin = min(kmin, lowz_key(a));
            kmax = max(kmax, lowz_key(b));
        }
    }
    kmin = __reduce_min_sync(0xffffffffu, kmin);
    kmax = __reduce_max_sync(0xffffffffu, kmax);
    if ((threadIdx.x & 31) == 0) {
        atomicMin(keys + 0, kmin);
        atomicMax(keys + 1, kmax);
    }
}

__global__ void lowz_band_kernel(const unsigned int *__restrict__ keys, float Zf, int n_xz, int n_yz, int *__restrict__ band)
{
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    const int N[2] = {n_xz, n_yz};
    const double Z = (double)Zf;
    double zl = 0.0, zh = -1.0;
    if (keys[0] <= keys[1]) { // some column is non-empty
        zl = (double)lowz_unkey(keys[0]);
        zh = (double)lowz_unkey(keys[1]);
        if (zl < 0.0) zl = 0.0;
        if (zh > Z) zh = Z;
    }
    for (int p = 0; p < 2; p++) {
        int b0 = 0, b1 = 0; // nothing can be fetched: one row is kept so that the array is not empty
        if (zl <= zh) {
            const double qa = __dsub_rn(__ddiv_rn(__dmul_rn(zl, (double)N[p]), Z), 0.515625); // - 1/2 - 1/64
            const double qb = __dsub_rn(__ddiv_rn(__dmul_rn(zh, (double)N[p]), Z), 0.484375); // - 1/2 + 1/64
            const long long a = (long long)floor(qa), b = (long long)floor(qb) + 1;
            b0 = (int)(a < 0 ? 0 : a);
            b1 = (int)(b > N[p] - 1 ? N[p] - 1 : b);
        }
        band[2 * p] = b0;
        band[2 * p + 1] = b1;
    }
}

// band[4] (HOST) = first/last kept z row of plane xz, then of plane yz.  Synchronises `st`.
int omerf_lowz_band(const omerf_scene *s, const float *d_lo, const float *d_up, int n_xz, int n_yz, int *band, cudaStream_t st)
{
    unsigned int *d_keys = nullptr;
    OMERF_CUDA(cudaMalloc((void **)&d_keys, 2 * sizeof(unsigned int) + 4 * sizeof(int)));
    const unsigned int init[2] = {0xffffffffu, 0u};
    cudaError_t e = cudaMemcpyAsync(d_keys, init, sizeof init, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) {
        const int n = s->dev.Mx * s->dev.My;
        lowz_bounds_kernel<<<(n + 1023) / 1024 < 1184 ? (n + 1023) / 1024 : 1184, 256, 0, st>>>(d_lo, d_up, n, d_keys);
        lowz_band_kernel<<<1, 32, 0, st>>>(d_keys, s->dev.box[2], n_xz, n_yz, (int *)(d_keys + 2));
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaMemcpyAsync(band, d_keys + 2, 4 * sizeof(int), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    cudaFree(d_keys);
    if (e != cudaSuccess) return omerf_cuda_fail(e, "low-z band");
    return OMERF_OK;
}

// ------------------------------------------------------------------------------------------ pyramid
__global__ void pyr_level0_kernel(const float *__restrict__ lo, const float *__restrict__ up,
                                  float2 *__restrict__ out, int n)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = make_float2(lo[i], up[i]);
}

__global__ void pyr_reduce_kernel(const float2 *__restrict__ src, int snx, int sny, float2 *__restrict__ dst,
                                  int dnx, int dny)
{
    int j = blockIdx.x * blockDim.x + threadIdx.x; // fast axis = y
    int i = blockIdx.y * blockDim.y + threadIdx.y;
    if (i >= dnx || j >= dny) return;
    float mn = INFINITY, mx = -INFINITY;
    for (int a = 0; a < 2; a++)
        for (int b = 0; b < 2; b++) {
            int si = 2 * i + a, sj = 2 * j + b;
            if (si < snx && sj < sny) {
                float2 v = src[(size_t)si * sny + sj];
                mn = fminf(mn, v.x);
                mx = fmaxf(mx, v.y);
            }
        }
    dst[(size_t)i * dny + j] = make_float2(mn, mx);
}

int omerf_launch_pyramid(omerf_scene *s, const float *d_lo, const float *d_up, cudaStream_t st)
{
    DevScene &v = s->dev;
    int nx = v.Mx, ny = v.My, L = 0;
    size_t total = 0;
    while (true) {
        v.lvl_nx[L] = nx;
        v.lvl_ny[L] = ny;
        v.lvl_off[L] = (int)total;
        total += (size_t)nx * ny;
        L++;
        if ((nx == 1 && ny == 1) || L == OMERF_MAX_LEVELS) break;
        nx = (nx + 1) / 2;
        ny = (ny + 1) / 2;
    }
    if (total > 0x7fffffffull) {
        omerf_set_error("invalid argument: occupancy plane too large");
        return OMERF_ERR_INVALID;
    }
    v.n_levels = L;
    v.n_pyr = (uint32_t)total;
    OMERF_CUDA(cudaMalloc(&s->d_pyr, total * sizeof(float2)));
    s->device_bytes += total * sizeof(float2);
    v.pyr = (const float2 *)s->d_pyr;
    float2 *pyr = (float2 *)s->d_pyr;
    int n0 = v.Mx * v.My;
    pyr_level0_kernel<<<(n0 + 255) / 256, 256, 0, st>>>(d_lo, d_up, pyr, n0);
    for (int l = 1; l < L; l++) {
        dim3 blk(32, 8), grd((v.lvl_ny[l] + 31) / 32, (v.lvl_nx[l] + 7) / 8);
        pyr_reduce_kernel<<<grd, blk, 0, st>>>(pyr + v.lvl_off[l - 1], v.lvl_nx[l - 1], v.lvl_ny[l - 1],
                                               pyr + v.lvl_off[l], v.lvl_nx[l], v.lvl_ny[l]);
    }
    OMERF_CUDA(cudaGetLastError());
    return OMERF_OK;
}

// ------------------------------------------------------------------------------------------ bitfield
// Cell i overlaps voxel j along one axis with positive length iff (exact integers)
//   2 j (M-1) < (2i+1) N   and   (2i-1) N < 2 (j+1) (M-1)
__device__ __forceinline__ void cell_range(int j, int N, int M, int *i0, int *i1)
{
    long long a = 2ll * j * (M - 1), e = 2ll * (j + 1) * (M - 1);
    // smallest i with (2i+1) N > a  <=>  i > (a/N - 1)/2
    long long lo = (a / N - 1) / 2 - 1;
    if (lo < 0) lo = 0;
    while (lo < M - 1 && !((2 * lo + 1) * N > a)) lo++;
    long long hi = lo;
    while (hi + 1 <= M - 1 && (2 * (hi + 1) - 1) * N < e) hi++;
    *i0 = (int)lo;
    *i1 = ((2 * lo + 1) * N > a && (2 * lo - 1) * N < e) ? (int)hi : (int)lo - 1;
}

__global__ void occ_level0_kernel(DevScene sc, uint32_t *__restrict__ out, unsigned long long n_words,
                                  unsigned long long n_bits)
{
    unsigned long long w = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (w >= n_words) return;
    const int Nx = sc.N[0], Ny = sc.N[1], Nz = sc.N[2];
    const double Z = (double)sc.box[2];
    uint32_t word = 0;
    int cjx = -1, cjy = -1, x0 = 0, x1 = -1, y0 = 0, y1 = -1;
    for (int b = 0; b < 32; b++) {
        unsigned long long idx = w * 32 + b;
        if (idx >= n_bits) break;
        int jz = (int)(idx % Nz);
        unsigned long long col = idx / Nz;
        int jy = (int)(col % Ny), jx = (int)(col / Ny);
        if (jx != cjx) {
            cell_range(jx, Nx, sc.Mx, &x0, &x1);
            cjx = jx;
        }
        if (jy != cjy) {
            cell_range(jy, Ny, sc.My, &y0, &y1);
            cjy = jy;
        }
        double zl = __ddiv_rn(__dmul_rn((double)jz, Z), (double)Nz);
        double zh = __ddiv_rn(__dmul_rn((double)(jz + 1), Z), (double)Nz);
        bool set = false;
        for (int ix = x0; ix <= x1 && !set; ix++)
            for (int iy = y0; iy <= y1 && !set; iy++) {
                float2 h = sc.pyr[(size_t)ix * sc.My + iy]; // level 0 = the field itself
                double lo = (double)h.x, hi = (double)h.y;
                if (lo <= hi && zl <= hi && zh >= lo) set = true;
            }
        if (set) word |= 1u << b;
    }
    out[w] = word;
}

__device__ __forceinline__ bool occ_bit(const uint32_t *bits, int ny, int nz, int jx, int jy, int jz)
{
    unsigned long long idx = ((unsigned long long)jx * ny + jy) * nz + jz;
    return (bits[idx >> 5] >> (idx & 31)) & 1u;
}

__global__ void occ_reduce_kernel(const uint32_t *__restrict__ src, int snx, int sny, int snz,
                                  uint32_t *__restrict__ dst, int dnx, int dny, int dnz,
                                  unsigned long long n_words, unsigned long long n_bits)
{
    unsigned long long w = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (w >= n_words) return;
    uint32_t word = 0;
    for (int b = 0; b < 32; b++) {
        unsigned long long idx = w * 32 + b;
        if (idx >= n_bits) break;
        int jz = (int)(idx % dnz);
        unsigned long long col = idx / dnz;
        int jy = (int)(col % dny), jx = (int)(col / dny);
        bool set = false;
        for (int a = 0; a < 2 && !set; a++)
            for (int c = 0; c < 2 && !set; c++)
                for (int e = 0; e < 2 && !set; e++) {
                    int x = 2 * jx + a, y = 2 * jy + c, z = 2 * jz + e;
                    if (x < snx && y < sny && z < snz) set = occ_bit(src, sny, snz, x, y, z);
                }
        if (set) word |= 1u << b;
    }
    dst[w] = word;
}

__global__ void popcount_kernel(const uint32_t *__restrict__ words, unsigned long long n_words,
                                unsigned long long *__restrict__ total)
{
    unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
    unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
    unsigned long long acc = 0;
    for (; i < n_words; i += stride) acc += __popc(words[i]);
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, o);
    if ((threadIdx.x & 31) == 0 && acc) atomicAdd(total, acc);
}

int omerf_launch_bitfield(omerf_scene *s, cudaStream_t st)
{
    DevScene &v = s->dev;
    int nx = v.N[0], ny = v.N[1], nz = v.N[2], L = 0;
    unsigned long long total_words = 0;
    while (true) {
        v.occ_nx[L] = nx;
        v.occ_ny[L] = ny;
        v.occ_nz[L] = nz;
        v.occ_off[L] = total_words;
        total_words += ((unsigned long long)nx * ny * nz + 31) / 32;
        L++;
        if ((nx == 1 && ny == 1 && nz == 1) || L == OMERF_MAX_LEVELS) break;
        nx = (nx + 1) / 2;
        ny = (ny + 1) / 2;
        nz = (nz + 1) / 2;
    }
    v.occ_levels = L;
    v.n_occ_words = total_words;
    OMERF_CUDA(cudaMalloc(&s->d_occ, total_words * 4 + 16));
    s->device_bytes += total_words * 4;
    v.occ = (const uint32_t *)s->d_occ;
    uint32_t *occ = (uint32_t *)s->d_occ;
    unsigned long long *d_total = (unsigned long long *)(occ + total_words + (total_words & 1));
    OMERF_CUDA(cudaMemsetAsync(d_total, 0, 8, st));
    unsigned long long bits0 = (unsigned long long)v.N[0] * v.N[1] * v.N[2];
    unsigned long long words0 = (bits0 + 31) / 32;
    occ_level0_kernel<<<(unsigned)((words0 + 127) / 128), 128, 0, st>>>(v, occ, words0, bits0);
    for (int l = 1; l < L; l++) {
        unsigned long long nb = (unsigned long long)v.occ_nx[l] * v.occ_ny[l] * v.occ_nz[l];
        unsigned long long nw = (nb + 31) / 32;
        occ_reduce_kernel<<<(unsigned)((nw + 127) / 128), 128, 0, st>>>(
            occ + v.occ_off[l - 1], v.occ_nx[l - 1], v.occ_ny[l - 1], v.occ_nz[l - 1], occ + v.occ_off[l],
            v.occ_nx[l], v.occ_ny[l], v.occ_nz[l], nw, nb);
    }
    popcount_kernel<<<1184, 256, 0, st>>>(occ, words0, d_total);
    OMERF_CUDA(cudaGetLastError());
    OMERF_CUDA(cudaMemcpyAsync(&s->occ_bits_set, d_total, 8, cudaMemcpyDeviceToHost, st));
    OMERF_CUDA(cudaStreamSynchronize(st));
    return OMERF_OK;
}

// ------------------------------------------------------------------------------------------ MLP weight packing
// G: 34 -> 16 -> 16 -> 3 (Eq. 4).  The render kernel evaluates it for 16 rays at a time with
// mma.sync.m16n8k8 (tf32 x 3 split: a_hi b_hi + a_lo b_hi + a_hi b_lo, fp32 accumulate), so the weights are
// stored once in B-fragment order: lane (g = lane/4, t = lane%4) of tile (k-step s, n-tile q) holds
//   layer 1:  W0[8q+g][8s+t],    W0[8q+g][8s+t+4]      (zero beyond the 34 inputs)
//   layer 2:  W1[8q+g][8s+2t],   W1[8q+g][8s+2t+1]     (k order = the C-fragment order of layer 1's output,
//   layer 3:  W2[g][8s+2t],      W2[g][8s+2t+1]         so hidden activations never leave their registers)
__device__ __forceinline__ float tf32_rna(float x)
{
    uint32_t r;
    asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(r) : "f"(x));
    return __uint_as_float(r);
}

__global__ void mlp_pack_kernel(const float *__restrict__ W0, const float *__restrict__ b0,
                                const float *__restrict__ W1, const float *__restrict__ b1,
                                const float *__restrict__ W2, const float *__restrict__ b2, float2 *__restrict__ tab)
{
    const int lane = threadIdx.x & 31, tile = threadIdx.x >> 5; // 21 warps: 16 weight tiles + 5 bias tiles
    const int g = lane >> 2, t = lane & 3;
    if (tile < OMERF_MLP_TILES) {
        float w0 = 0.0f, w1 = 0.0f;
        if (tile < 10) {
            // layer-1 columns are permuted (omerf_mlp.cuh: mlp_orig_of_col); padding columns carry weight 0
            const int s = tile >> 1, q = tile & 1, n = 8 * q + g, k0 = mlp_orig_of_col(8 * s + t), k1 = mlp_orig_of_col(8 * s + t + 4);
            if (k0 >= 0) w0 = W0[n * OMERF_MLP_IN + k0];
            if (k1 >= 0) w1 = W0[n * OMERF_MLP_IN + k1];
        } else if (tile < 14) {
            const int s = (tile - 10) >> 1, q = (tile - 10) & 1, n = 8 * q + g;
            w0 = W1[n * OMERF_MLP_HID + 8 * s + 2 * t];
            w1 = W1[n * OMERF_MLP_HID + 8 * s + 2 * t + 1];
        } else {
            const int s = tile - 14;
            if (g < 3) {
                w0 = W2[g * OMERF_MLP_HID + 8 * s + 2 * t];
                w1 = W2[g * OMERF_MLP_HID + 8 * s + 2 * t + 1];
            }
        }
        const float h0 = tf32_rna(w0), h1 = tf32_rna(w1);
        tab[(tile * 2 + 0) * 32 + lane] = make_float2(h0, h1);
        tab[(tile * 2 + 1) * 32 + lane] = make_float2(tf32_rna(w0 - h0), tf32_rna(w1 - h1));
    } else {
        const int bt = tile - OMERF_MLP_TILES; // C-fragment columns 2t, 2t+1 of n-tile
        float v0 = 0.0f, v1 = 0.0f;
        if (bt < 2) {
            v0 = b0[8 * bt + 2 * t];
            v1 = b0[8 * bt + 2 * t + 1];
        } else if (bt < 4) {
            v0 = b1[8 * (bt - 2) + 2 * t];
            v1 = b1[8 * (bt - 2) + 2 * t + 1];
        } else {
            if (2 * t < 3) v0 = b2[2 * t];
            if (2 * t + 1 < 3) v1 = b2[2 * t + 1];
        }
        tab[OMERF_MLP_BIAS_OFF + bt * 32 + lane] = make_float2(v0, v1);
    }
}

int omerf_launch_mlp_pack(omerf_scene *s, const omerf_scene_desc *d, cudaStream_t st)
{
    const int nW0 = OMERF_MLP_HID * OMERF_MLP_IN, nW1 = OMERF_MLP_HID * OMERF_MLP_HID, nW2 = 3 * OMERF_MLP_HID;
    const int total = nW0 + nW1 + nW2 + 2 * OMERF_MLP_HID + 3;
    float host[OMERF_MLP_HID * OMERF_MLP_IN + OMERF_MLP_HID * OMERF_MLP_HID + 3 * OMERF_MLP_HID + 2 * OMERF_MLP_HID + 3];
    float *p = host;
    memcpy(p, d->W0, nW0 * 4); p += nW0;
    memcpy(p, d->b0, OMERF_MLP_HID * 4); p += OMERF_MLP_HID;
    memcpy(p, d->W1, nW1 * 4); p += nW1;
    memcpy(p, d->b1, OMERF_MLP_HID * 4); p += OMERF_MLP_HID;
    memcpy(p, d->W2, nW2 * 4); p += nW2;
    memcpy(p, d->b2, 3 * 4);
    float *raw = nullptr;
    OMERF_CUDA(cudaMalloc((void **)&raw, total * 4));
    cudaError_t e = cudaMemcpyAsync(raw, host, total * 4, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaMalloc(&s->d_mlp_tab, OMERF_MLP_TAB_LEN * sizeof(float2));
    if (e == cudaSuccess) {
        const float *W0 = raw, *b0 = W0 + nW0, *W1 = b0 + OMERF_MLP_HID, *b1 = W1 + nW1, *W2 = b1 + OMERF_MLP_HID, *b2 = W2 + nW2;
        mlp_pack_kernel<<<1, 32 * (OMERF_MLP_TILES + 5), 0, st>>>(W0, b0, W1, b1, W2, b2, (float2 *)s->d_mlp_tab);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    cudaFree(raw);
    if (e != cudaSuccess) return omerf_cuda_fail(e, "MLP weight packing");
    s->dev.mlp_tab = (const float2 *)s->d_mlp_tab;
    s->device_bytes += OMERF_MLP_TAB_LEN * sizeof(float2);
    return OMERF_OK;
}

// ------------------------------------------------------------------------------------------ S9: sample-count heat map
__global__ void heatmap_kernel(const uint32_t *__restrict__ n, unsigned long long n_pixels, uint32_t n_max, uint8_t *__restrict__ out)
{
    const unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_pixels) return;
    const uint32_t c = min(n[i], n_max);
    const int v = (int)((unsigned long long)c * 255ull / n_max);
    out[i * 3 + 0] = (uint8_t)v;
    out[i * 3 + 1] = (uint8_t)(255 - abs(2 * v - 255));
    out[i * 3 + 2] = (uint8_t)(255 - v);
}

int omerf_launch_heatmap(const uint32_t *n, unsigned long long n_pixels, uint32_t n_max, uint8_t *out, cudaStream_t st)
{
    if (n_pixels == 0) return OMERF_OK;
    const unsigned long long blocks = (n_pixels + 255) / 256;
    if (blocks > 0x7fffffffull) {
        omerf_set_error("invalid argument: too many pixels");
        return OMERF_ERR_INVALID;
    }
    heatmap_kernel<<<(unsigned int)blocks, 256, 0, st>>>(n, n_pixels, n_max, out);
    OMERF_CUDA(cudaGetLastError());
    return OMERF_OK;
}
