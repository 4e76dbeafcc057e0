// omerf_device.cuh — device-side scene description shared by the scene-build and render kernels.
// Internal to the CUDA path (never included by oracle/).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/omerf.h"

#define OMERF_MAX_LEVELS 16
#define OMERF_MLP_IN 34
#define OMERF_MLP_HID 16
#define OMERF_MLP_TILES 16
#define OMERF_MLP_BIAS_OFF (OMERF_MLP_TILES * 2 * 32)
#define OMERF_MLP_TAB_LEN (OMERF_MLP_BIAS_OFF + 5 * 32)

// Column order of the deferred MLP's layer-1 input matrix (explained in omerf_mlp.cuh): column -> input index of Eq. 4
// in the order of DESIGN.md R13 (-1: padding column, weight 0), and its inverse.
__host__ __device__ constexpr inline int mlp_orig_of_col(int col)
{
    const int s = col >> 3, r = col & 7, t = r & 3, i = 2 * s + (r >> 2);
    if (t == 3) return i < 4 ? 3 + i : -1;
    if (i == 0) return 7 + t;
    if (i == 9) return t;
    return 10 + (3 * ((i - 1) >> 1) + t) * 2 + ((i - 1) & 1);
}
__host__ __device__ constexpr inline int mlp_col(int j) // inverse: the column that holds input j
{
    for (int col = 0; col < 40; col++)
        if (mlp_orig_of_col(col) == j) return col;
    return -1;
}


// Everything a render kernel needs, passed by value as a __grid_constant__ kernel parameter, so scalars, sizes and
// pointers are read through the constant bank.  The deferred MLP's weights are not in here: they sit in global memory
// in tensor-core fragment order (mlp_tab below) and are read with __ldg by mma_x3 / mlp_tiles (omerf_mlp.cuh).
struct DevScene {
    float box[3];
    // occupancy plane P_o and its min/max pyramid ("2D max pooling")
    int Mx, My;
    float sx, sy;          // (Mx-1)/X, (My-1)/Y in fp32: the predicate's scale (Eq. 7 nearest grid point)
    float cell_x, cell_y;  // X/(Mx-1): world size of a cell, proposals only
    int n_levels;
    const float2 *pyr;     // all levels, (min of h_lo, max of h_up) per node, [nx][ny] row-major
    int lvl_off[OMERF_MAX_LEVELS], lvl_nx[OMERF_MAX_LEVELS], lvl_ny[OMERF_MAX_LEVELS];
    // features: 8 uint8 channels per texel = 8 bytes; every array ENTRY is a pair of texels adjacent along ONE axis of the
    // array, (t[i], t[min(i+1, N-1)]), with the bytes of the two texels interleaved channel by channel (pair_entry below):
    // one 16-byte load brings both taps of that axis, already in the operand order of the IDP.2A dot products (S0 layout).
    // Paired axis: y for V, the second axis for the planes.
    int G[3];
    float gs[3];           // G/box per axis
    const uint4 *grid;     // dense: [Gx][Gy][Gz] entries (pairs along y); sparse blocks: atlas [id][B][B][B] (omerf_sparse.cu)
    int blk_shift;         // 0 = dense grid, else log2 of the block edge B
    int nby, nbz;          // block-grid dims along y and z
    const int32_t *blk_table; // [nbx][nby][nbz] block id or -1
    int xy_n[2], xz_n[2], yz_n[2];
    float xy_s[2], xz_s[2], yz_s[2];
    const uint4 *pxy, *pxz, *pyz; // [A][B] entries, pairs along the second axis
    int xz_rows, yz_rows;  // stored entries per row of xz / yz: the z band kept by the low-z bake (= xz_n[1] without it)
    int xz_zoff, yz_zoff;  // first stored z row ("low resolution in the z direction, according to the upper and
                           // lower bounds of the occupancy plane"; R27)
    int shared_taps;       // xy_n[0] == xz_n[0], xy_n[1] == yz_n[0], xz_n[1] == yz_n[1]: three taps serve the six plane axes
    float deq_mul, deq_add; // scale/65536, 4*bias
    float deq_mul_half, deq_add_half; // halves of the two: the per-sample sigmoids take tanh of half the pre-activation
    float step, inv_step;
    uint32_t q_stop;
    float bg[3];
    float soft_eps, inv_soft_eps; // > 0: Eq. 6 soft occupancy weights the colour contributions (Eq. 8)
    // sampler GRID (config-4 comparator): multi-resolution binary occupancy grid
    int sampler;
    int N[3];
    float ns[3];           // N/box per axis
    float vox[3];          // box/N per axis (proposals only)
    int occ_levels;
    const uint32_t *occ;   // all levels; level l has dims ceil(N/2^l), bit index ((jx*ny+jy)*nz+jz)
    unsigned long long occ_off[OMERF_MAX_LEVELS]; // word offset of each level
    int occ_nx[OMERF_MAX_LEVELS], occ_ny[OMERF_MAX_LEVELS], occ_nz[OMERF_MAX_LEVELS];
    // deferred MLP G (Eq. 4): weights pre-arranged as mma.m16n8k8 B fragments, split into tf32 hi + lo
    // (omerf_build.cu: mlp_pack_kernel).  tab[(tile*2 + part)*32 + lane], part 0 = hi, 1 = lo; tiles 0..9 layer 1
    // (k-step*2 + n-tile), 10..13 layer 2, 14..15 layer 3; then 5 bias tiles (layer 1 n-tiles 0,1; layer 2; layer 3).
    const float2 *mlp_tab;
    // element counts of the arrays above, for the range checks of the OMERF_CHECKED build (omerf_render.cu)
    uint32_t n_pyr, n_grid, n_pxy, n_pxz, n_pyz, n_blk;
    unsigned long long n_occ_words;
};

// S0 entry of two texels a, b (8 channels each): bytes (a.c0, b.c0, a.c1, b.c1 | a.c2, b.c2, a.c3, b.c3 | ... c4..c7)
__device__ __forceinline__ uint4 pair_entry(uint2 a, uint2 b)
{
    return make_uint4(__byte_perm(a.x, b.x, 0x5140), __byte_perm(a.x, b.x, 0x7362), __byte_perm(a.y, b.y, 0x5140),
                      __byte_perm(a.y, b.y, 0x7362));
}

struct omerf_scene {
    DevScene dev;
    int device;
    void *d_pyr, *d_grid, *d_pxy, *d_pxz, *d_pyz, *d_occ, *d_mlp_tab, *d_blk_table;
    uint64_t blocks_total, blocks_allocated, grid_bytes, plane_bytes;
    int band[4];           // first/last stored z row of plane xz, then of plane yz
    uint64_t device_bytes;
    uint64_t occ_bits_set;
    // per-render state (mutable through the const handle: calls must be stream-ordered)
    mutable omerf_camera *d_cams;
    mutable omerf_camera *h_cams;      // pinned staging ring
    mutable cudaEvent_t *slot_event;
    mutable int cam_capacity;          // views per slot
    mutable unsigned long long call_index;
    mutable float *d_scratch_rgb;
    mutable uint32_t *d_scratch_n;
    mutable uint64_t scratch_pixels;
    mutable int last_launches;
    mutable cudaStream_t copy_stream;  // omerf_render_host: copies a band back while the next one renders
    mutable cudaEvent_t band_event[16];
    // omerf_render_host_async: two scratch sets used in turn; async_done[i] = the copy-back out of set i has finished
    mutable float *d_async_rgb[2];
    mutable uint32_t *d_async_n[2];
    mutable uint64_t async_pixels;
    mutable cudaEvent_t async_done[2];
    mutable unsigned long long async_index;
    unsigned int *d_tile_counter;     // work-queue heads of the persistent march kernel, one per camera-ring slot
    int persistent_blocks;            // resident CTAs of the march kernel (SMs x occupancy)
};

#define OMERF_CAM_SLOTS 16
#define OMERF_COUNTER_WORDS 64   // per ring slot: word 0 = work-queue head, word 32 = logged samples (calibration render)

// error plumbing (omerf_api.cu)
void omerf_set_error(const char *fmt, ...);
int omerf_cuda_fail(cudaError_t e, const char *what);
#define OMERF_CUDA(call)                                                     \
    do {                                                                     \
        cudaError_t e__ = (call);                                            \
        if (e__ != cudaSuccess) return omerf_cuda_fail(e__, #call);          \
    } while (0)

// kernels' host launchers
int omerf_launch_pyramid(omerf_scene *s, const float *d_lo, const float *d_up, cudaStream_t st);
int omerf_launch_bitfield(omerf_scene *s, cudaStream_t st);
int omerf_launch_pair_layout(const void *d_src, void *d_dst, unsigned long long total, int n, unsigned long long stride, cudaStream_t st);
int omerf_lowz_band(const omerf_scene *s, const float *d_lo, const float *d_up, int n_xz, int n_yz, int *band, cudaStream_t st);
int omerf_bake_sparse_grid(omerf_scene *s, void **d_dense, int block, cudaStream_t st);
int omerf_launch_mlp_pack(omerf_scene *s, const omerf_scene_desc *d, cudaStream_t st);
int omerf_launch_render(const omerf_scene *s, const omerf_camera *d_cams, int n_views, int W, int H,
                        float *out_rgb, uint32_t *out_n, cudaStream_t st, unsigned int *tile_counter, int *launches,
                        uint2 *sample_log = nullptr,
                        unsigned int log_capacity = 0, unsigned int tile_first = 0, unsigned int tile_end = 0);
int omerf_launch_gather_probe(const omerf_scene *s, const omerf_camera *d_cam, int W, const uint2 *sample_log,
                              unsigned int n, unsigned int mult, uint32_t *sink, cudaStream_t st);
int omerf_query_persistent_blocks(int sampler, int *blocks);
int omerf_launch_heatmap(const uint32_t *n, unsigned long long n_pixels, uint32_t n_max, uint8_t *out, cudaStream_t st);
int omerf_launch_smoothness(const omerf_scene *s, long long n, int S, const float *F, const float *dir, const float *delta,
                            float *out_loss, float *out_G, cudaStream_t st);
