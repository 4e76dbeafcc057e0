/*
 * omerf.h — C-ABI of the B200-native Oblique-MERF renderer (arxiv 2404.09531).
 *
 * The boundary follows the paper's problem statement: baked assets + camera -> image
 * (PAPER.md:186-188 sec. 4.4, :79-81 Eq. 4) and BASELINE.json:north_star's entry points.
 * Plain pointers and sizes only; every pointer is marked HOST or DEVICE.  All work
 * (layout, pyramid, ray generation, marching, gathers, compositing, MLP) runs in
 * hand-written CUDA kernels for sm_100a; there is no CPU fallback.
 *
 * Conventions:
 *   world box [0,X]x[0,Y]x[0,Z], z up.  Host arrays are C-contiguous, first
 *   named axis slowest, channel last.  Channel 0 = density, 1..3 = diffuse RGB,
 *   4..7 = specular features (Eq. 3).
 *   Pixel (u,v): row v = 0 is the TOP row, centre (u+0.5, v+0.5); the ray through it is
 *   normalize(fwd + ((u+0.5-cx)/fx) right - ((v+0.5-cy)/fy) up); right/up/fwd orthonormal.
 *
 * Errors: every int-returning call returns OMERF_OK (0) or a negative code and never throws or
 * aborts; omerf_last_error() gives a thread-local message for the last failure.
 */
#ifndef OMERF_H
#define OMERF_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define OMERF_OK 0
#define OMERF_ERR_INVALID (-1) /* null pointer, non-positive size, step <= 0, t_stop not in (0,1), mlp shape */
#define OMERF_ERR_NOMEM (-2)   /* out of device memory */
#define OMERF_ERR_CUDA (-3)    /* any other CUDA failure (message in omerf_last_error) */

#define OMERF_SAMPLER_PLANE 0 /* occupancy-plane march — the method */
#define OMERF_SAMPLER_GRID 1  /* binary occupancy-grid DDA (the structure PAPER.md:188 replaces; BASELINE.json configs[4]) */

typedef struct omerf_scene omerf_scene; /* opaque; owns all device memory of one baked scene */

/* Baked scene on the HOST.  omerf_scene_create deep-copies everything; on the device every feature array
 * is re-laid out as 16-byte entries of two adjacent texels (twice the host bytes; omerf_scene_info.device_bytes). */
typedef struct {
    float box[3];      /* X, Y, Z */
    int32_t hf_n[2];   /* Mx, My: grid points of the occupancy plane P_o; vertex-centred, spacing X/(Mx-1) */
    const float *h_lo; /* HOST [Mx][My] z_min */
    const float *h_up; /* HOST [Mx][My] z_max; h_up < h_lo marks an empty column */
    int32_t grid_n[3]; /* Gx, Gy, Gz */
    const uint8_t *grid; /* HOST [Gx][Gy][Gz][8] low-res voxel grid V */
    int32_t xy_n[2], xz_n[2], yz_n[2];
    const uint8_t *plane_xy; /* HOST [Ax][Ay][8], sampled with (x,y) */
    const uint8_t *plane_xz; /* HOST [Ax][Az][8], sampled with (x,z) */
    const uint8_t *plane_yz; /* HOST [Ay][Az][8], sampled with (y,z) */
    float deq_scale, deq_bias; /* pre-activation of one source = u8*deq_scale + deq_bias (28/255, -14) */
    int32_t mlp_in, mlp_hidden; /* must be 34 and 16: G is 34 -> 16 -> 16 -> 3 (Eq. 4) */
    const float *W0, *b0, *W1, *b1, *W2, *b2; /* HOST, row-major [out][in] */
    float step;     /* sample spacing delta along the ray (world units) */
    float t_stop;   /* early-termination transmittance, in (0,1) */
    float bg[3];    /* background colour */
    int32_t sampler; /* OMERF_SAMPLER_PLANE or OMERF_SAMPLER_GRID */
    int32_t occ_n[3]; /* sampler GRID: bitfield resolution (e.g. 2048,2048,256); derived on the device from the slab */
    float soft_eps;   /* 0: binary mask (render time).  > 0, sampler PLANE only: the soft occupancy
                         function M of Eq. 6 (q = 2) with buffer zones of height soft_eps weights every
                         sample's colour contribution, C = sum_i M_i w_i c_i (Eq. 8) - the training-time
                         forward pass.  Samples, transmittance and termination are those of the binary mask; where the
                         two buffers of a thin interval overlap the smaller ramp is taken (R23). */
    int32_t grid_block; /* 0: V is stored dense.  2, 4, 8 or 16: V is stored as sparse blocks of grid_block^3 voxels
                            baked on the device from the occupancy plane: only blocks
                           holding a voxel that a sample inside the slab can touch are kept (R24); the
                           rendered images are identical to the dense layout's.  Sampler PLANE only: the grid sampler's
                           voxels are a superset of the slab (OMERF_ERR_INVALID otherwise). */
    int32_t lowz_bake;  /* 0: plane_xz / plane_yz are stored whole.  1: low-z bake ("a texture map with high
                           resolution in the xy direction and low resolution in the z direction, according to the upper
                           and lower bounds of the occupancy plane"): only the band of z rows that a sample inside
                           [min z_min, max z_max] of the occupancy plane can touch is uploaded and stored (DESIGN.md
                           R27); the rendered images are identical.  Sampler PLANE only. */
} omerf_scene_desc;

/* Pinhole camera, world frame. */
typedef struct {
    float origin[3], right[3], up[3], fwd[3];
    float fx, fy, cx, cy; /* pixels */
} omerf_camera;

typedef struct {
    uint64_t device_bytes;  /* device memory held by the scene (features + occupancy structures) */
    int32_t pyramid_levels; /* levels of the min/max pyramid of (h_lo, h_up), level 0 = P_o itself */
    int32_t sampler;
    uint64_t occ_bits_set;  /* sampler GRID: number of set voxels of the derived bitfield, else 0 */
    uint64_t grid_bytes;        /* device bytes of V: dense array, or atlas + block table */
    uint64_t grid_blocks_total; /* sparse layout: blocks of the block grid, else 0 */
    uint64_t grid_blocks_allocated; /* sparse layout: blocks kept (occupancy ratio = allocated / total, cf. Table 5) */
    uint64_t plane_bytes;       /* device bytes of the three planes (cf. the VRAM column of Table 3) */
    int32_t xz_band[2], yz_band[2]; /* first and last z row of plane_xz / plane_yz that is stored (the whole plane without
                                       lowz_bake) */
} omerf_scene_info;

/* S0 + S1 (+ S10 derivation): validate, upload, re-lay out for gathers, build the min/max pyramid
 * ("2D max pooling to obtain multiple low-resolution occupancy planes") and, for
 * sampler GRID, the occupancy bitfield.  Synchronous; on return the caller may free every host array.
 * The scene is immutable afterwards. */
int omerf_scene_create(const omerf_scene_desc *desc /*HOST*/, omerf_scene **out_scene);

/* S2..S9: render n_views images of W x H pixels (PAPER.md:188 marching; Eq. 1-4, 7-8).
 *   cameras       HOST  [n_views]; read before the call returns
 *   out_rgb       DEVICE [n_views][H][W][3] float32, 4-byte aligned
 *   out_nsamples  DEVICE [n_views][H][W] uint32: samples fetched per pixel (Fig. 1)
 *   stream        cudaStream_t (NULL = default stream)
 * Asynchronous: kernels are enqueued on `stream`; results are valid once the caller has synchronised it.
 * Threads and streams: a scene handle keeps per-call state (a 16-slot ring of pinned camera staging, device cameras
 * and work-queue heads, the launch counter, the scratch of omerf_render_host), so it must NOT be used by two host
 * threads at once - serialise the calls (one thread at a time).  Serialised calls may use different streams: a ring slot
 * is reused only after the kernel that last used it has finished (the 17th call in flight waits for the 1st).
 * The scene's device must be the current device (else OMERF_ERR_INVALID).
 * Allocation: the first call with more views than any call before it re-allocates the camera ring
 * (cudaDeviceSynchronize + cudaMalloc inside the call); calls after that warm-up do not allocate. */
int omerf_render(const omerf_scene *scene, const omerf_camera *cameras /*HOST*/, int n_views, int W, int H,
                 float *out_rgb /*DEVICE*/, uint32_t *out_nsamples /*DEVICE*/, void *stream);

/* A share of the same work (pixels and views are independent, the scene is read-only, so a batch is
 * partitioned across GPUs with no exchange): renders only the 8x4-pixel tiles [tile_first, tile_end) of the batch, tiles
 * numbered view-major, then row-major inside a view (tiles_x = ceil(W/8), tiles_y = ceil(H/4)).  out_rgb / out_nsamples
 * are the FULL batch buffers; pixels of other tiles are not written.  tile_first <= tile_end <= n_views*tiles_x*tiles_y
 * (else OMERF_ERR_INVALID); an empty range is a no-op.  Everything else as omerf_render. */
int omerf_render_tiles(const omerf_scene *scene, const omerf_camera *cameras /*HOST*/, int n_views, int W, int H,
                       float *out_rgb /*DEVICE*/, uint32_t *out_nsamples /*DEVICE*/, uint32_t tile_first,
                       uint32_t tile_end, void *stream);

/* Same path with HOST outputs (pinned or pageable): renders into scene-owned device scratch on
 * `stream` in bands of whole tile rows, copies each band back on a scene-owned second stream while the next
 * band renders, and synchronises both streams before returning.  The first call with more pixels than any call
 * before it (re)allocates the scratch (cudaDeviceSynchronize + cudaMalloc inside the call).  Same threading rule as
 * omerf_render. */
int omerf_render_host(const omerf_scene *scene, const omerf_camera *cameras /*HOST*/, int n_views, int W,
                      int H, float *out_rgb /*HOST*/, uint32_t *out_nsamples /*HOST*/, void *stream);

/* Pipelined form of omerf_render_host (SURVEY.md 8(b) "Async"): the same banded render + copy-back, but the call returns
 * as soon as the work is enqueued, so the copy-back of frame N overlaps the render of frame N + 1 (a frame's 16 B per pixel
 * take longer to cross PCIe than to render).  Two scene-owned scratch sets alternate between calls; a set is rendered
 * into again only after its previous copy-back has finished (event-ordered on the device, the host never blocks).
 *   out_rgb / out_nsamples  HOST, as omerf_render_host.  They belong to the library from this call until omerf_wait
 *                           returns: do not read, reuse or free them before.  PINNED memory is needed for the overlap; with
 *                           pageable buffers the result is the same but cudaMemcpyAsync blocks the call.
 *   cameras                 HOST, read before the call returns.
 * Calls on one scene complete in call order.  The first call with more pixels than any async call before it (re)allocates
 * both scratch sets (cudaDeviceSynchronize + cudaMalloc inside the call).  Same threading rule as omerf_render; use one
 * `stream` for consecutive calls, or order the streams yourself.
 * omerf_wait blocks the host until every omerf_render_host_async call made on this scene so far has delivered its host
 * buffers (OMERF_OK also when there was none). */
int omerf_render_host_async(const omerf_scene *scene, const omerf_camera *cameras /*HOST*/, int n_views, int W, int H,
                            float *out_rgb /*HOST*/, uint32_t *out_nsamples /*HOST*/, void *stream);
int omerf_wait(const omerf_scene *scene);

/* omerf_render for callers that must not allocate.  omerf_render keeps its per-call scratch - the device copy of the
 * cameras and the head of the march kernel's work queue - in a ring it (re)allocates with cudaMalloc / cudaMallocHost
 * behind a cudaDeviceSynchronize whenever a call brings more views than any call before it.  That is wrong for two kinds
 * of caller: a render or serving loop with a frame deadline (an allocation synchronises the whole device and stalls every
 * other stream of the process, at a moment the loop does not choose), and a plug-in inside a host program that has
 * already claimed all device memory for its own pool or forbids driver allocations once start-up is over (cudaMalloc then
 * fails, or breaks the host's memory accounting).  This entry point renders the same images with the same march kernel,
 * but the kernel's scratch lives in ONE fixed array that is part of the library image: a file-scope __device__ array of
 * 256 B (queue head) + OMERF_STATIC_MAX_VIEWS * 64 B (cameras) = 2304 B, which every GPU that loads the library holds
 * until the process exits.  It calls no cudaMalloc, cudaMallocHost, cudaFree or any other allocating routine; the scene
 * handle (an input, made earlier by whoever may allocate) and both outputs are still the caller's.
 *   cameras       HOST [n_views], 0 <= n_views <= OMERF_STATIC_MAX_VIEWS (more: OMERF_ERR_INVALID with a message that
 *                 names the limit; split the batch, or use omerf_render).  Passed to the GPU as launch arguments, so the
 *                 array may be pageable and may be reused or freed as soon as the call returns.
 *   out_rgb, out_nsamples, W, H, stream: as omerf_render.  There is no limit on W or H.
 * Set-up: the first call on each device looks up the device address of the array (cudaGetSymbolAddress, with that device
 * current) and keeps it; make that first call before any stream capture begins.  Later calls only launch.
 * Sharing: there is one array per GPU, shared by every scene, stream and thread.  Calls are safe back to back on one
 * stream (each call clears the queue head and rewrites the cameras in stream order; nothing is carried over from the
 * previous call).  Two calls whose kernels can overlap on the GPU - different streams without an ordering between them -
 * RACE on the array and give wrong images; order them with an event, or use omerf_render for one of them (its scratch
 * is separate).  Same one-host-thread-per-scene rule as omerf_render; asynchronous on `stream`. */
#define OMERF_STATIC_MAX_VIEWS 32
int omerf_render_static(const omerf_scene *scene, const omerf_camera *cameras /*HOST*/, int n_views, int W, int H,
                        float *out_rgb /*DEVICE*/, uint32_t *out_nsamples /*DEVICE*/, void *stream);

/* Gather calibration (SURVEY.md 8(d) "L2/L1 gather rate": the builder must calibrate the achievable rate of the
 * same load width over the same footprint).  Renders one frame of `camera` while logging every sample taken, then
 * times a kernel that only replays the feature loads of Eq. 2 for those samples - the 10 sixteen-byte
 * entries (pairs of adjacent texels) that hold a sample's 20 texels in the scene's device layout - with no filtering,
 * activations or compositing, once in frame order (pixel-coherent addresses) and once in a scattered order.  A sample
 * needs 160 B of distinct texels.  flush_l2 != 0 overwrites a 256 MiB buffer before every timed launch.
 * Synchronous (device-wide); owns and frees its scratch.  HOST pointers. */
typedef struct {
    uint64_t samples;       /* samples of the frame (= sum of out_nsamples) */
    double ms_frame_order;  /* mean duration of one replay launch, frame order */
    double ms_scattered;    /* mean duration of one replay launch, scattered order */
} omerf_gather_probe_result;
int omerf_gather_probe(const omerf_scene *scene, const omerf_camera *camera /*HOST, one view*/, int W, int H,
                       int repeats, int flush_l2, omerf_gather_probe_result *out /*HOST*/);

/* View-direction smoothness term, forward pass (Eq. 9-10): for each of n viewing
 * directions d_i with deferred-shading input F_i = [sum w c^d (3), sum w f (4)] (Eq. 4) and S perturbations delta_is
 * (the caller's draws from N(0, Sigma), Eq. 9),
 *     out_loss[i] = sum_s cos(d_i, d_i + delta_is) * || G(F_i, d_i + delta_is) - G(F_i, d_i) ||_2^2       (Eq. 10)
 * with the scene's deferred MLP G.  The perturbed direction enters the encoding as it is (R25).
 *   F DEVICE float32 [n][7], dir DEVICE [n][3], delta DEVICE [n][S][3], out_loss DEVICE [n],
 *   out_G DEVICE [n][S+1][3] (row 0 = G(F,d)) or NULL.  Asynchronous on `stream`; n >= 0, S >= 0. */
int omerf_mlp_smoothness(const omerf_scene *scene, int64_t n, int S, const float *F /*DEVICE*/,
                         const float *dir /*DEVICE*/, const float *delta /*DEVICE*/, float *out_loss /*DEVICE*/,
                         float *out_G /*DEVICE or NULL*/, void *stream);

/* Sample-count visualisation (Fig. 1, "number of samples"; S9 of SURVEY.md 8(a)): maps per-pixel sample
 * counts to an 8-bit colour ramp from blue (0 samples) over green to red (>= n_max samples), in exact integers:
 *     v = min(n, n_max) * 255 / n_max,   rgb = (v, 255 - |2 v - 255|, 255 - v).
 * The paper prints no colour map; this ramp is the repo's choice (R26).
 *   nsamples DEVICE uint32 [n_pixels], out_rgb8 DEVICE uint8 [n_pixels][3]; n_max >= 1; asynchronous on `stream`. */
int omerf_heatmap(const uint32_t *nsamples /*DEVICE*/, uint64_t n_pixels, uint32_t n_max, uint8_t *out_rgb8 /*DEVICE*/,
                  void *stream);

/* Number of kernels of this library the last omerf_render / omerf_render_host on this scene launched. */
int omerf_last_launch_count(const omerf_scene *scene);

int omerf_scene_get_info(const omerf_scene *scene, omerf_scene_info *out_info /*HOST*/);

/* Test hooks: copy derived structures back to the HOST (synchronous).
 * level in [0, pyramid_levels): out_min/out_max HOST [nx][ny] float32 with nx = ceil(Mx / 2^level);
 * *nx, *ny receive the level's size; pass out_min = out_max = NULL to query the size only. */
int omerf_scene_get_pyramid_level(const omerf_scene *scene, int level, int32_t *nx, int32_t *ny,
                                  float *out_min /*HOST*/, float *out_max /*HOST*/);
/* sparse layout: out_table HOST int32[n] with n = grid_blocks_total, C order of (bx,by,bz); block id or -1. */
int omerf_scene_get_block_table(const omerf_scene *scene, int32_t *out_table /*HOST*/, uint64_t n);
/* sampler GRID: out_words HOST uint32[(Nx*Ny*Nz+31)/32], bit index ((jx*Ny + jy)*Nz + jz), LSB first. */
int omerf_scene_get_bitfield(const omerf_scene *scene, uint32_t *out_words /*HOST*/, uint64_t n_words);

void omerf_scene_destroy(omerf_scene *scene); /* NULL is a no-op */

const char *omerf_last_error(void); /* thread-local, static storage; "" if none */
const char *omerf_version(void);
/* Diagnostic of the range-checked build (libomerf_checked.so: every device index of the render kernels is checked, a
 * violation is redirected to element 0 and recorded).  In that build it synchronises the device, returns the bit mask of
 * violations seen since the last call (bit: 0 pyramid, 1 V, 2 xy, 3 xz, 4 yz, 5 block table, 6 bitfield, 7 view, 8 pixel,
 * 9 pool slot, 10 pool list; 0xffffffff: CUDA error) and clears it.  The shipped library compiles the checks away: there
 * the call touches no CUDA state (no synchronisation) and returns 0. */
unsigned int omerf_check_errors(void);

#ifdef __cplusplus
}
#endif
#endif /* OMERF_H */
