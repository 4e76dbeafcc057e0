// omerf_api.cu — host side of the C-ABI (include/omerf.h): validation, upload, ownership, errors.
// No rendering arithmetic lives here; every step of the path runs in the kernels of
// omerf_build.cu (S0/S1/S10 derivations) and omerf_render.cu (S2..S9).
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <string.h>

#include <new>

#include "omerf_device.cuh"

static thread_local char g_err[512] = "";

void omerf_set_error(const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof g_err, fmt, ap);
    va_end(ap);
}

int omerf_cuda_fail(cudaError_t e, const char *what)
{
    omerf_set_error("CUDA error %d (%s) in %s", (int)e, cudaGetErrorString(e), what);
    cudaGetLastError(); // clear the sticky-less error state
    return e == cudaErrorMemoryAllocation ? OMERF_ERR_NOMEM : OMERF_ERR_CUDA;
}

extern "C" const char *omerf_last_error(void) { return g_err; }
extern "C" const char *omerf_version(void) { return "omerf-b200 0.1 (sm_100a)"; }

static int invalid(const char *msg)
{
    omerf_set_error("invalid argument: %s", msg);
    return OMERF_ERR_INVALID;
}

static int upload(void **dptr, const void *host, size_t bytes, uint64_t *total)
{
    OMERF_CUDA(cudaMalloc(dptr, bytes));
    OMERF_CUDA(cudaMemcpy(*dptr, host, bytes, cudaMemcpyHostToDevice));
    *total += bytes;
    return OMERF_OK;
}

static void free_scene(omerf_scene *s)
{
    if (!s) return;
    cudaFree(s->d_pyr);
    cudaFree(s->d_grid);
    cudaFree(s->d_pxy);
    cudaFree(s->d_pxz);
    cudaFree(s->d_pyz);
    cudaFree(s->d_occ);
    cudaFree(s->d_mlp_tab);
    cudaFree(s->d_blk_table);
    cudaFree(s->d_cams);
    cudaFree(s->d_tile_counter);
    cudaFree(s->d_scratch_rgb);
    cudaFree(s->d_scratch_n);
    for (int i = 0; i < 2; i++) {
        cudaFree(s->d_async_rgb[i]);
        cudaFree(s->d_async_n[i]);
        if (s->async_done[i]) cudaEventDestroy(s->async_done[i]);
    }
    if (s->h_cams) cudaFreeHost(s->h_cams);
    if (s->copy_stream) {
        cudaStreamDestroy(s->copy_stream);
        for (int i = 0; i < 16; i++)
            if (s->band_event[i]) cudaEventDestroy(s->band_event[i]);
    }
    if (s->slot_event) {
        for (int i = 0; i < OMERF_CAM_SLOTS; i++)
            if (s->slot_event[i]) cudaEventDestroy(s->slot_event[i]);
        delete[] s->slot_event;
    }
    delete s;
}

extern "C" int omerf_scene_create(const omerf_scene_desc *d, omerf_scene **out_scene)
{
    g_err[0] = 0;
    if (!d || !out_scene) return invalid("null desc/out_scene");
    *out_scene = nullptr;
    if (!(d->box[0] > 0 && d->box[1] > 0 && d->box[2] > 0)) return invalid("box must be positive");
    if (d->hf_n[0] < 2 || d->hf_n[1] < 2) return invalid("hf_n must be >= 2");
    if (!d->h_lo || !d->h_up) return invalid("null height field");
    for (int i = 0; i < 3; i++)
        if (d->grid_n[i] < 1) return invalid("grid_n must be >= 1");
    for (int i = 0; i < 2; i++)
        if (d->xy_n[i] < 1 || d->xz_n[i] < 1 || d->yz_n[i] < 1) return invalid("plane sizes must be >= 1");
    // the gather takes index and weight of a tap from one conversion, exact for fewer than 2^15 texels per axis
    {
        const int32_t dims[] = {d->grid_n[0], d->grid_n[1], d->grid_n[2], d->xy_n[0], d->xy_n[1], d->xz_n[0], d->xz_n[1], d->yz_n[0], d->yz_n[1]};
        for (int32_t n : dims)
            if (n > (1 << 15)) return invalid("a feature array has more than 32768 texels along an axis");
    }
    // the gather addresses texels with 32-bit indices
    if ((unsigned long long)d->grid_n[0] * d->grid_n[1] * d->grid_n[2] > 0xffffffffull ||
        (unsigned long long)d->xy_n[0] * d->xy_n[1] > 0xffffffffull || (unsigned long long)d->xz_n[0] * d->xz_n[1] > 0xffffffffull ||
        (unsigned long long)d->yz_n[0] * d->yz_n[1] > 0xffffffffull)
        return invalid("a feature array has more than 2^32 - 1 texels");
    if (!d->grid || !d->plane_xy || !d->plane_xz || !d->plane_yz) return invalid("null feature array");
    if (d->mlp_in != OMERF_MLP_IN || d->mlp_hidden != OMERF_MLP_HID) return invalid("MLP must be 34 -> 16 -> 16 -> 3");
    if (!d->W0 || !d->b0 || !d->W1 || !d->b1 || !d->W2 || !d->b2) return invalid("null MLP array");
    if (!(d->step > 0) || !isfinite(d->step)) return invalid("step must be > 0");
    if (!(d->t_stop > 0 && d->t_stop < 1)) return invalid("t_stop must be in (0,1)");
    if (d->sampler != OMERF_SAMPLER_PLANE && d->sampler != OMERF_SAMPLER_GRID) return invalid("unknown sampler");
    if (d->grid_block != 0 && d->grid_block != 2 && d->grid_block != 4 && d->grid_block != 8 && d->grid_block != 16)
        return invalid("grid_block must be 0, 2, 4, 8 or 16");
    if (!(d->soft_eps >= 0) || !isfinite(d->soft_eps)) return invalid("soft_eps must be >= 0");
    if (d->soft_eps > 0 && d->sampler != OMERF_SAMPLER_PLANE) return invalid("soft_eps needs the occupancy-plane sampler");
    // the sparse-block bake (R24) keeps what a sample INSIDE THE SLAB can touch; the grid sampler's voxels are a superset of the
    // slab (R18), so its samples may have corners in blocks that were not kept
    if (d->grid_block != 0 && d->sampler != OMERF_SAMPLER_PLANE) return invalid("grid_block needs the occupancy-plane sampler");
    if (d->lowz_bake != 0 && d->lowz_bake != 1) return invalid("lowz_bake must be 0 or 1");
    if (d->lowz_bake && d->sampler != OMERF_SAMPLER_PLANE) return invalid("lowz_bake needs the occupancy-plane sampler");
    if (d->sampler == OMERF_SAMPLER_GRID)
        for (int i = 0; i < 3; i++)
            if (d->occ_n[i] < 1) return invalid("occ_n must be >= 1 for the grid sampler");

    omerf_scene *s = new (std::nothrow) omerf_scene();
    if (!s) {
        omerf_set_error("host allocation failed");
        return OMERF_ERR_NOMEM;
    }
    memset(s, 0, sizeof *s);
    if (cudaGetDevice(&s->device) != cudaSuccess) {
        int rc = omerf_cuda_fail(cudaGetLastError(), "cudaGetDevice (no CUDA device: there is no CPU fallback)");
        delete s;
        return rc;
    }
    DevScene &v = s->dev;
    for (int i = 0; i < 3; i++) v.box[i] = d->box[i];
    v.Mx = d->hf_n[0];
    v.My = d->hf_n[1];
    v.sx = (float)(v.Mx - 1) / d->box[0];
    v.sy = (float)(v.My - 1) / d->box[1];
    v.cell_x = d->box[0] / (float)(v.Mx - 1);
    v.cell_y = d->box[1] / (float)(v.My - 1);
    for (int i = 0; i < 3; i++) {
        v.G[i] = d->grid_n[i];
        v.gs[i] = (float)d->grid_n[i] / d->box[i];
    }
    const int ax[3][2] = {{0, 1}, {0, 2}, {1, 2}};
    const int32_t *pn[3] = {d->xy_n, d->xz_n, d->yz_n};
    int *vn[3] = {v.xy_n, v.xz_n, v.yz_n};
    float *vs[3] = {v.xy_s, v.xz_s, v.yz_s};
    for (int p = 0; p < 3; p++)
        for (int i = 0; i < 2; i++) {
            vn[p][i] = pn[p][i];
            vs[p][i] = (float)pn[p][i] / d->box[ax[p][i]];
        }
    v.shared_taps = d->xy_n[0] == d->xz_n[0] && d->xy_n[1] == d->yz_n[0] && d->xz_n[1] == d->yz_n[1];
    v.deq_mul = d->deq_scale / 65536.0f;
    v.deq_add = 4.0f * d->deq_bias;
    v.deq_mul_half = 0.5f * v.deq_mul;
    v.deq_add_half = 0.5f * v.deq_add;
    v.step = d->step;
    v.inv_step = 1.0f / d->step;
    v.q_stop = (uint32_t)ceil(-log((double)d->t_stop) * 1048576.0);
    for (int i = 0; i < 3; i++) v.bg[i] = d->bg[i];
    v.sampler = d->sampler;
    v.soft_eps = d->soft_eps;
    v.inv_soft_eps = d->soft_eps > 0 ? 1.0f / d->soft_eps : 0.0f;

    int rc = OMERF_OK;
    float *d_lo = nullptr, *d_up = nullptr;
    void *d_raw = nullptr; // raw texels of the array being laid out
    uint64_t tmp = 0;
    size_t hf_bytes = (size_t)v.Mx * v.My * sizeof(float);
    do {
        // S1: min/max pyramid of the two height fields, built on the device
        if ((rc = upload((void **)&d_lo, d->h_lo, hf_bytes, &tmp))) break;
        if ((rc = upload((void **)&d_up, d->h_up, hf_bytes, &tmp))) break;
        if ((rc = omerf_launch_pyramid(s, d_lo, d_up, 0))) break;
        // 8(f).1: z band of the xz / yz planes kept by the low-z bake (the whole plane without it)
        s->band[0] = s->band[2] = 0;
        s->band[1] = v.xz_n[1] - 1;
        s->band[3] = v.yz_n[1] - 1;
        if (d->lowz_bake && (rc = omerf_lowz_band(s, d_lo, d_up, v.xz_n[1], v.yz_n[1], s->band, 0))) break;
        v.xz_zoff = s->band[0];
        v.xz_rows = s->band[1] - s->band[0] + 1;
        v.yz_zoff = s->band[2];
        v.yz_rows = s->band[3] - s->band[2] + 1;
        // S0: features.  8 channels per texel = 8 bytes; stored as 16-byte entries of two texels adjacent along y (V) or the
        // second axis (planes) (omerf_build.cu: pair_layout_kernel).  Only the kept z band of xz / yz is uploaded at all.
        struct {
            const uint8_t *host;
            size_t rows;
            int n_host, first, n;
            void **dst;
        } arr[4] = {{d->grid, (size_t)v.G[0] * v.G[1], v.G[2], 0, v.G[2], &s->d_grid},
                    {d->plane_xy, (size_t)v.xy_n[0], v.xy_n[1], 0, v.xy_n[1], &s->d_pxy},
                    {d->plane_xz, (size_t)v.xz_n[0], v.xz_n[1], v.xz_zoff, v.xz_rows, &s->d_pxz},
                    {d->plane_yz, (size_t)v.yz_n[0], v.yz_n[1], v.yz_zoff, v.yz_rows, &s->d_pyz}};
        // The raw texels of a dense array never sit on the device as a whole: the destination (2x) is allocated first and
        // the source passes through a staging buffer of at most OMERF_STAGE_BYTES, a whole number of pairing units at a time
        // (a unit holds both texels of every pair: an x slab of V, one row of a plane), so the peak of scene_create is the
        // resident layout plus one staging buffer instead of plus the whole raw array.
        const size_t OMERF_STAGE_BYTES = (size_t)64 << 20;
        for (int a = 0; a < 4 && rc == OMERF_OK; a++) {
            const size_t raw_bytes = arr[a].rows * arr[a].n * 8;
            cudaError_t e;
            if (a == 0 && d->grid_block) {
                // 8(f).1: sparse-block layout of V baked from the occupancy plane (takes the whole raw array, frees it)
                e = cudaMalloc(&d_raw, raw_bytes);
                if (e == cudaSuccess) e = cudaMemcpy(d_raw, arr[a].host, raw_bytes, cudaMemcpyHostToDevice);
                if (e != cudaSuccess) {
                    rc = omerf_cuda_fail(e, "feature upload");
                    break;
                }
                s->d_grid = d_raw;
                d_raw = nullptr;
                rc = omerf_bake_sparse_grid(s, &s->d_grid, d->grid_block, 0);
                s->device_bytes += s->grid_bytes;
                continue;
            }
            if ((e = cudaMalloc(arr[a].dst, raw_bytes * 2)) != cudaSuccess) {
                rc = omerf_cuda_fail(e, "feature layout");
                break;
            }
            const size_t row_bytes = (size_t)arr[a].n * 8;
            const size_t unit_rows = a == 0 ? (size_t)v.G[1] : 1, n_units = arr[a].rows / unit_rows;
            size_t units_per_chunk = OMERF_STAGE_BYTES / (unit_rows * row_bytes);
            units_per_chunk = units_per_chunk < 1 ? 1 : (units_per_chunk > n_units ? n_units : units_per_chunk);
            if ((e = cudaMalloc(&d_raw, units_per_chunk * unit_rows * row_bytes)) != cudaSuccess) {
                rc = omerf_cuda_fail(e, "feature staging");
                break;
            }
            for (size_t u0 = 0; u0 < n_units && rc == OMERF_OK; u0 += units_per_chunk) {
                const size_t k = n_units - u0 < units_per_chunk ? n_units - u0 : units_per_chunk;
                const size_t r0 = u0 * unit_rows, nr = k * unit_rows;
                // a pageable copy on the null stream: ordered behind the kernel that still reads the buffer
                e = cudaMemcpy2D(d_raw, row_bytes, arr[a].host + (r0 * (size_t)arr[a].n_host + (size_t)arr[a].first) * 8,
                                 (size_t)arr[a].n_host * 8, row_bytes, nr, cudaMemcpyHostToDevice);
                if (e != cudaSuccess) {
                    rc = omerf_cuda_fail(e, "feature upload");
                    break;
                }
                uint4 *dst = (uint4 *)*arr[a].dst + r0 * (size_t)arr[a].n;
                if (a == 0) rc = omerf_launch_pair_layout(d_raw, dst, nr * arr[a].n, v.G[1], (unsigned long long)v.G[2], 0);
                else rc = omerf_launch_pair_layout(d_raw, dst, nr * arr[a].n, arr[a].n, 1ull, 0);
            }
            if (rc) break;
            if ((e = cudaDeviceSynchronize()) != cudaSuccess) {
                rc = omerf_cuda_fail(e, "feature layout");
                break;
            }
            cudaFree(d_raw);
            d_raw = nullptr;
            s->device_bytes += raw_bytes * 2;
            if (a == 0) s->grid_bytes = raw_bytes * 2;
            else s->plane_bytes += raw_bytes * 2;
        }
        if (rc) break;
        if (!d->grid_block) {
            v.grid = (const uint4 *)s->d_grid;
            v.n_grid = (uint32_t)((size_t)v.G[0] * v.G[1] * v.G[2]);
        }
        v.n_pxy = (uint32_t)((size_t)v.xy_n[0] * v.xy_n[1]);
        v.n_pxz = (uint32_t)((size_t)v.xz_n[0] * v.xz_rows);
        v.n_pyz = (uint32_t)((size_t)v.yz_n[0] * v.yz_rows);
        v.pxy = (const uint4 *)s->d_pxy;
        v.pxz = (const uint4 *)s->d_pxz;
        v.pyz = (const uint4 *)s->d_pyz;
        // S0: deferred-MLP weights -> tensor-core fragment order, tf32 hi/lo split (device kernel)
        if ((rc = omerf_launch_mlp_pack(s, d, 0))) break;
        // S10: occupancy bitfield + its mip chain, derived on the device from the slab
        if (d->sampler == OMERF_SAMPLER_GRID) {
            for (int i = 0; i < 3; i++) {
                v.N[i] = d->occ_n[i];
                v.ns[i] = (float)d->occ_n[i] / d->box[i];
                v.vox[i] = d->box[i] / (float)d->occ_n[i];
            }
            if ((rc = omerf_launch_bitfield(s, 0))) break;
        }
        cudaError_t e = cudaDeviceSynchronize();
        if (e != cudaSuccess) {
            rc = omerf_cuda_fail(e, "scene build");
            break;
        }
        if ((rc = omerf_query_persistent_blocks(d->sampler, &s->persistent_blocks))) break;
        {
            // one work-queue head per camera-ring slot (word 0; word 32 counts logged samples in the calibration render)
            cudaError_t ee = cudaMalloc((void **)&s->d_tile_counter, OMERF_CAM_SLOTS * OMERF_COUNTER_WORDS * sizeof(unsigned int));
            if (ee != cudaSuccess) {
                rc = omerf_cuda_fail(ee, "cudaMalloc tile counter");
                break;
            }
        }
        // camera staging ring
        s->cam_capacity = 0;
        s->slot_event = new (std::nothrow) cudaEvent_t[OMERF_CAM_SLOTS]();
        if (!s->slot_event) {
            omerf_set_error("host allocation failed");
            rc = OMERF_ERR_NOMEM;
            break;
        }
        for (int i = 0; i < OMERF_CAM_SLOTS && rc == OMERF_OK; i++) {
            cudaError_t ee = cudaEventCreateWithFlags(&s->slot_event[i], cudaEventDisableTiming);
            if (ee != cudaSuccess) rc = omerf_cuda_fail(ee, "cudaEventCreate");
        }
    } while (0);
    cudaFree(d_lo);
    cudaFree(d_up);
    cudaFree(d_raw);
    if (rc != OMERF_OK) {
        free_scene(s);
        return rc;
    }
    *out_scene = s;
    return OMERF_OK;
}

extern "C" void omerf_scene_destroy(omerf_scene *s)
{
    if (!s) return;
    cudaDeviceSynchronize();
    free_scene(s);
}

static int ensure_cams(const omerf_scene *s, int n_views)
{
    if (n_views <= s->cam_capacity) return OMERF_OK;
    OMERF_CUDA(cudaDeviceSynchronize()); // kernels of earlier calls still read the ring that is about to be freed
    cudaFree(s->d_cams);
    if (s->h_cams) cudaFreeHost(s->h_cams);
    s->d_cams = nullptr;
    s->h_cams = nullptr;
    s->cam_capacity = 0;
    int cap = n_views < 16 ? 16 : n_views;
    size_t bytes = (size_t)cap * OMERF_CAM_SLOTS * sizeof(omerf_camera);
    OMERF_CUDA(cudaMalloc((void **)&s->d_cams, bytes));
    OMERF_CUDA(cudaMallocHost((void **)&s->h_cams, bytes));
    s->cam_capacity = cap;
    return OMERF_OK;
}

// the scene's device must be the current one: every pointer in the handle belongs to it
static int check_device(const omerf_scene *s)
{
    int dev = -1;
    OMERF_CUDA(cudaGetDevice(&dev));
    if (dev != s->device) {
        omerf_set_error("invalid argument: scene lives on device %d but device %d is current", s->device, dev);
        return OMERF_ERR_INVALID;
    }
    return OMERF_OK;
}

// Stages the cameras and launches the march kernel for the tiles [tile_first, tile_end) of the batch (0, 0 = all).
// *slot_io: ring slot of an earlier band of the same call (-1: take the next slot and stage the cameras now).
// A slot (pinned staging, device cameras, work-queue head) is reused only after the last kernel that used it has
// finished: its event is recorded after the launch.
static int render_impl(const omerf_scene *s, const omerf_camera *cameras, int n_views, int W, int H, float *out_rgb,
                       uint32_t *out_nsamples, void *stream, unsigned int tile_first, unsigned int tile_end, int *slot_io)
{
    if (!s || !cameras || !out_rgb || !out_nsamples) return invalid("null scene/cameras/output");
    if (n_views < 0 || W <= 0 || H <= 0) return invalid("n_views >= 0, W > 0, H > 0 required");
    if (((uintptr_t)out_rgb & 3) || ((uintptr_t)out_nsamples & 3)) return invalid("misaligned output");
    if (n_views == 0) return OMERF_OK;
    cudaStream_t st = (cudaStream_t)stream;
    int rc = check_device(s);
    if (rc) return rc;
    if ((rc = ensure_cams(s, n_views))) return rc;
    int slot = slot_io ? *slot_io : -1;
    if (slot < 0) {
        // stage the cameras: user memory -> pinned ring slot -> device ring slot (stream-ordered)
        slot = (int)(s->call_index++ % OMERF_CAM_SLOTS);
        OMERF_CUDA(cudaEventSynchronize(s->slot_event[slot]));
        omerf_camera *h = s->h_cams + (size_t)slot * s->cam_capacity;
        memcpy(h, cameras, (size_t)n_views * sizeof(omerf_camera));
        OMERF_CUDA(cudaMemcpyAsync(s->d_cams + (size_t)slot * s->cam_capacity, h, (size_t)n_views * sizeof(omerf_camera),
                                   cudaMemcpyHostToDevice, st));
        if (slot_io) *slot_io = slot;
    }
    int launches = 0;
    rc = omerf_launch_render(s, s->d_cams + (size_t)slot * s->cam_capacity, n_views, W, H, out_rgb, out_nsamples, st,
                             s->d_tile_counter + (size_t)slot * OMERF_COUNTER_WORDS, &launches, nullptr, 0, tile_first, tile_end);
    s->last_launches += launches;
    if (rc) return rc;
    OMERF_CUDA(cudaEventRecord(s->slot_event[slot], st));
    return OMERF_OK;
}

extern "C" int omerf_render(const omerf_scene *s, const omerf_camera *cameras, int n_views, int W, int H,
                            float *out_rgb, uint32_t *out_nsamples, void *stream)
{
    if (s) s->last_launches = 0;
    return render_impl(s, cameras, n_views, W, H, out_rgb, out_nsamples, stream, 0, 0, nullptr);
}

extern "C" int omerf_render_tiles(const omerf_scene *s, const omerf_camera *cameras, int n_views, int W, int H,
                                  float *out_rgb, uint32_t *out_nsamples, uint32_t tile_first, uint32_t tile_end, void *stream)
{
    if (W > 0 && H > 0 && n_views >= 0) {
        const unsigned long long all = (unsigned long long)((W + 7) / 8) * ((H + 3) / 4) * (unsigned long long)n_views;
        if (tile_first > tile_end || tile_end > all) return invalid("tile range must satisfy first <= end <= tiles of the batch");
    }
    if (s) s->last_launches = 0;
    if (tile_first == tile_end && s && cameras && out_rgb && out_nsamples && W > 0 && H > 0 && n_views >= 0) return OMERF_OK;
    return render_impl(s, cameras, n_views, W, H, out_rgb, out_nsamples, stream, tile_first, tile_end, nullptr);
}

extern "C" int omerf_render_host(const omerf_scene *s, const omerf_camera *cameras, int n_views, int W, int H,
                                 float *out_rgb, uint32_t *out_nsamples, void *stream)
{
    if (!s || !cameras || !out_rgb || !out_nsamples) return invalid("null scene/cameras/output");
    if (n_views < 0 || W <= 0 || H <= 0) return invalid("n_views >= 0, W > 0, H > 0 required");
    if (n_views == 0) return OMERF_OK;
    {
        int rc = check_device(s);
        if (rc) return rc;
    }
    uint64_t px = (uint64_t)n_views * W * H;
    if (px > s->scratch_pixels) {
        OMERF_CUDA(cudaDeviceSynchronize());
        cudaFree(s->d_scratch_rgb);
        cudaFree(s->d_scratch_n);
        s->d_scratch_rgb = nullptr;
        s->d_scratch_n = nullptr;
        s->scratch_pixels = 0;
        OMERF_CUDA(cudaMalloc((void **)&s->d_scratch_rgb, px * 3 * sizeof(float)));
        OMERF_CUDA(cudaMalloc((void **)&s->d_scratch_n, px * sizeof(uint32_t)));
        s->scratch_pixels = px;
    }
    cudaStream_t st = (cudaStream_t)stream;
    // The batch is rendered in bands of whole tile rows (one launch each, stream-ordered); a band is copied back on a
    // second stream while the next one renders.  Bands hold at least 10 MiB of output so that the fixed cost of a
    // launch (about 0.08 ms on B200) stays small against the copy it hides (1080p: 3 bands, 1.02 ms against 1.23 ms).
    if (!s->copy_stream) {
        OMERF_CUDA(cudaStreamCreateWithFlags(&s->copy_stream, cudaStreamNonBlocking));
        for (int i = 0; i < 16; i++) OMERF_CUDA(cudaEventCreateWithFlags(&s->band_event[i], cudaEventDisableTiming));
    }
    const unsigned int tiles_x = (unsigned int)((W + 7) / 8), tiles_y = (unsigned int)((H + 3) / 4);
    const uint64_t tile_rows = (uint64_t)n_views * tiles_y, out_bytes = px * 16;
    int bands = (int)(out_bytes / ((uint64_t)10 << 20));
    bands = bands < 1 ? 1 : (bands > 16 ? 16 : bands);
    if ((uint64_t)bands > tile_rows) bands = (int)tile_rows;
    auto pixel_row = [&](uint64_t R) { // first flattened pixel row (view * H + v) of flattened tile row R
        const uint64_t view = R / tiles_y, ty = R % tiles_y;
        const uint64_t v = ty * 4 < (uint64_t)H ? ty * 4 : (uint64_t)H;
        return view * (uint64_t)H + v;
    };
    s->last_launches = 0;
    int slot = -1;
    for (int b = 0; b < bands; b++) {
        const uint64_t R0 = tile_rows * b / bands, R1 = tile_rows * (b + 1) / bands;
        int rc = render_impl(s, cameras, n_views, W, H, s->d_scratch_rgb, s->d_scratch_n, stream, (unsigned int)(R0 * tiles_x),
                             (unsigned int)(R1 * tiles_x), &slot);
        if (rc) return rc;
        OMERF_CUDA(cudaEventRecord(s->band_event[b], st));
        OMERF_CUDA(cudaStreamWaitEvent(s->copy_stream, s->band_event[b], 0));
        const uint64_t r0 = pixel_row(R0), r1 = R1 == tile_rows ? (uint64_t)n_views * H : pixel_row(R1);
        OMERF_CUDA(cudaMemcpyAsync(out_rgb + r0 * W * 3, s->d_scratch_rgb + r0 * W * 3, (r1 - r0) * W * 3 * sizeof(float),
                                   cudaMemcpyDeviceToHost, s->copy_stream));
        OMERF_CUDA(cudaMemcpyAsync(out_nsamples + r0 * W, s->d_scratch_n + r0 * W, (r1 - r0) * W * sizeof(uint32_t),
                                   cudaMemcpyDeviceToHost, s->copy_stream));
    }
    OMERF_CUDA(cudaStreamSynchronize(s->copy_stream));
    OMERF_CUDA(cudaStreamSynchronize(st));
    return OMERF_OK;
}

// Pipelined form: the loop of omerf_render_host into one of two scratch sets, without the final synchronisation.  The render
// stream waits (on the device) for the previous copy-back out of the set it is about to overwrite; the copy stream runs the
// copies of consecutive calls in call order, so waiting for it (omerf_wait) is waiting for every host buffer.
extern "C" int omerf_render_host_async(const omerf_scene *s, const omerf_camera *cameras, int n_views, int W, int H,
                                       float *out_rgb, uint32_t *out_nsamples, void *stream)
{
    if (!s || !cameras || !out_rgb || !out_nsamples) return invalid("null scene/cameras/output");
    if (n_views < 0 || W <= 0 || H <= 0) return invalid("n_views >= 0, W > 0, H > 0 required");
    if (n_views == 0) return OMERF_OK;
    {
        int rc = check_device(s);
        if (rc) return rc;
    }
    const uint64_t px = (uint64_t)n_views * W * H;
    if (px > s->async_pixels) {
        OMERF_CUDA(cudaDeviceSynchronize());
        s->async_pixels = 0;
        for (int i = 0; i < 2; i++) {
            cudaFree(s->d_async_rgb[i]);
            cudaFree(s->d_async_n[i]);
            s->d_async_rgb[i] = nullptr;
            s->d_async_n[i] = nullptr;
        }
        for (int i = 0; i < 2; i++) {
            OMERF_CUDA(cudaMalloc((void **)&s->d_async_rgb[i], px * 3 * sizeof(float)));
            OMERF_CUDA(cudaMalloc((void **)&s->d_async_n[i], px * sizeof(uint32_t)));
            if (!s->async_done[i]) OMERF_CUDA(cudaEventCreateWithFlags(&s->async_done[i], cudaEventDisableTiming));
        }
        s->async_pixels = px;
    }
    if (!s->copy_stream) {
        OMERF_CUDA(cudaStreamCreateWithFlags(&s->copy_stream, cudaStreamNonBlocking));
        for (int i = 0; i < 16; i++) OMERF_CUDA(cudaEventCreateWithFlags(&s->band_event[i], cudaEventDisableTiming));
    }
    cudaStream_t st = (cudaStream_t)stream;
    const int set = (int)(s->async_index++ & 1ull);
    float *d_rgb = s->d_async_rgb[set];
    uint32_t *d_n = s->d_async_n[set];
    OMERF_CUDA(cudaStreamWaitEvent(st, s->async_done[set], 0)); // a never-recorded event counts as finished
    const unsigned int tiles_x = (unsigned int)((W + 7) / 8), tiles_y = (unsigned int)((H + 3) / 4);
    const uint64_t tile_rows = (uint64_t)n_views * tiles_y, out_bytes = px * 16;
    // Bands only shorten the fill of the pipeline (the first copy starts before the whole batch is rendered); in steady state
    // the overlap comes from the next call.  Every band is a launch with a fixed cost of about 0.08 ms, so bands are coarser
    // than omerf_render_host's: at least 32 MiB of output each (one 1080p frame: a single launch, 0.71 -> 0.61 ms per frame).
    int bands = (int)(out_bytes / ((uint64_t)32 << 20));
    bands = bands < 1 ? 1 : (bands > 16 ? 16 : bands);
    if ((uint64_t)bands > tile_rows) bands = (int)tile_rows;
    auto pixel_row = [&](uint64_t R) {
        const uint64_t view = R / tiles_y, ty = R % tiles_y;
        const uint64_t v = ty * 4 < (uint64_t)H ? ty * 4 : (uint64_t)H;
        return view * (uint64_t)H + v;
    };
    s->last_launches = 0;
    int slot = -1;
    for (int b = 0; b < bands; b++) {
        const uint64_t R0 = tile_rows * b / bands, R1 = tile_rows * (b + 1) / bands;
        int rc = render_impl(s, cameras, n_views, W, H, d_rgb, d_n, stream, (unsigned int)(R0 * tiles_x), (unsigned int)(R1 * tiles_x), &slot);
        if (rc) return rc;
        // a band event may be re-recorded by the next call while this wait is pending: a wait refers to the record before it
        OMERF_CUDA(cudaEventRecord(s->band_event[b], st));
        OMERF_CUDA(cudaStreamWaitEvent(s->copy_stream, s->band_event[b], 0));
        const uint64_t r0 = pixel_row(R0), r1 = R1 == tile_rows ? (uint64_t)n_views * H : pixel_row(R1);
        OMERF_CUDA(cudaMemcpyAsync(out_rgb + r0 * W * 3, d_rgb + r0 * W * 3, (r1 - r0) * W * 3 * sizeof(float), cudaMemcpyDeviceToHost,
                                   s->copy_stream));
        OMERF_CUDA(cudaMemcpyAsync(out_nsamples + r0 * W, d_n + r0 * W, (r1 - r0) * W * sizeof(uint32_t), cudaMemcpyDeviceToHost,
                                   s->copy_stream));
    }
    OMERF_CUDA(cudaEventRecord(s->async_done[set], s->copy_stream));
    return OMERF_OK;
}

extern "C" int omerf_wait(const omerf_scene *s)
{
    if (!s) return invalid("null scene");
    if (s->copy_stream) OMERF_CUDA(cudaStreamSynchronize(s->copy_stream));
    return OMERF_OK;
}


// Gather calibration: logs the samples of one frame, then times kernels that only replay their
// 10 entry loads (20 texels), in frame order and in a scattered order.  Synchronous; allocates and frees its own buffers.
extern "C" int omerf_gather_probe(const omerf_scene *s, const omerf_camera *camera, int W, int H, int repeats,
                                  int flush_l2, omerf_gather_probe_result *out)
{
    if (!s || !camera || !out) return invalid("null scene/camera/out");
    if (W <= 0 || H <= 0 || repeats <= 0) return invalid("W > 0, H > 0, repeats > 0 required");
    memset(out, 0, sizeof *out);
    const uint64_t px = (uint64_t)W * H;
    int rc = check_device(s);
    if (rc) return rc;
    if ((rc = ensure_cams(s, 1))) return rc;
    OMERF_CUDA(cudaDeviceSynchronize());
    omerf_camera *dv = s->d_cams; // slot 0 of the ring; nothing is in flight after the synchronise
    OMERF_CUDA(cudaMemcpy(dv, camera, sizeof(omerf_camera), cudaMemcpyHostToDevice));
    float *rgb = nullptr;
    uint32_t *cnt = nullptr, *sink = nullptr;
    uint2 *log = nullptr;
    char *flush = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    const size_t flush_bytes = (size_t)256 << 20;
    unsigned int cap = (unsigned int)(px * 8 < 0xffffffffull ? px * 8 : 0xffffffffull), n = 0;
    do {
        cudaError_t e;
#define PROBE_CUDA(call)                                       \
    if ((e = (call)) != cudaSuccess) {                         \
        rc = omerf_cuda_fail(e, #call);                        \
        break;                                                 \
    }
        PROBE_CUDA(cudaMalloc((void **)&rgb, px * 3 * sizeof(float)));
        PROBE_CUDA(cudaMalloc((void **)&cnt, px * sizeof(uint32_t)));
        for (int attempt = 0; attempt < 2 && rc == OMERF_OK; attempt++) {
            PROBE_CUDA(cudaMalloc((void **)&log, (size_t)cap * sizeof(uint2)));
            int launches = 0;
            if ((rc = omerf_launch_render(s, dv, 1, W, H, rgb, cnt, 0, s->d_tile_counter, &launches, log, cap))) break;
            PROBE_CUDA(cudaMemcpy(&n, s->d_tile_counter + 32, sizeof n, cudaMemcpyDeviceToHost));
            if (n <= cap) break;
            cudaFree(log); // more samples than the first guess: size the log exactly and log again
            log = nullptr;
            cap = n;
        }
        if (rc) break;
        out->samples = n;
        if (n == 0) break;
        PROBE_CUDA(cudaMalloc((void **)&sink, (size_t)n * sizeof(uint32_t)));
        if (flush_l2) PROBE_CUDA(cudaMalloc((void **)&flush, flush_bytes));
        PROBE_CUDA(cudaEventCreate(&e0));
        PROBE_CUDA(cudaEventCreate(&e1));
        // a multiplier coprime with n permutes the log; 1 keeps frame order
        unsigned int mult = 2654435761u % n;
        if (mult < 2) mult = 1;
        auto gcd = [](unsigned a, unsigned b) { while (b) { unsigned t = a % b; a = b; b = t; } return a; };
        while (mult > 1 && gcd(mult, n) != 1) mult--;
        for (int order = 0; order < 2 && rc == OMERF_OK; order++) {
            double total = 0.0;
            for (int it = -1; it < repeats && rc == OMERF_OK; it++) { // it = -1: warm-up
                if (flush) PROBE_CUDA(cudaMemsetAsync(flush, it & 0xff, flush_bytes, 0));
                PROBE_CUDA(cudaEventRecord(e0, 0));
                if ((rc = omerf_launch_gather_probe(s, dv, W, log, n, order ? mult : 1u, sink, 0))) break;
                PROBE_CUDA(cudaEventRecord(e1, 0));
                PROBE_CUDA(cudaEventSynchronize(e1));
                float ms = 0.f;
                PROBE_CUDA(cudaEventElapsedTime(&ms, e0, e1));
                if (it >= 0) total += ms;
            }
            (order ? out->ms_scattered : out->ms_frame_order) = total / repeats;
        }
#undef PROBE_CUDA
    } while (0);
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    cudaFree(rgb);
    cudaFree(cnt);
    cudaFree(log);
    cudaFree(sink);
    cudaFree(flush);
    return rc;
}

extern "C" int omerf_mlp_smoothness(const omerf_scene *s, int64_t n, int S, const float *F, const float *dir,
                                    const float *delta, float *out_loss, float *out_G, void *stream)
{
    if (!s) return invalid("null scene");
    if (n < 0 || S < 0) return invalid("n >= 0 and S >= 0 required");
    if (n == 0) return OMERF_OK;
    if (!F || !dir || !out_loss || (S > 0 && !delta)) return invalid("null F/dir/delta/out_loss");
    if ((unsigned long long)n * (unsigned long long)(S + 1) > 0x7fffffffffffull) return invalid("batch too large");
    {
        int rc = check_device(s);
        if (rc) return rc;
    }
    s->last_launches = 1;
    return omerf_launch_smoothness(s, n, S, F, dir, delta, out_loss, out_G, (cudaStream_t)stream);
}

extern "C" int omerf_heatmap(const uint32_t *nsamples, uint64_t n_pixels, uint32_t n_max, uint8_t *out_rgb8, void *stream)
{
    if (n_pixels == 0) return OMERF_OK;
    if (!nsamples || !out_rgb8) return invalid("null nsamples/out_rgb8");
    if (n_max < 1) return invalid("n_max must be >= 1");
    return omerf_launch_heatmap(nsamples, n_pixels, n_max, out_rgb8, (cudaStream_t)stream);
}

extern "C" int omerf_last_launch_count(const omerf_scene *s) { return s ? s->last_launches : 0; }

extern "C" int omerf_scene_get_info(const omerf_scene *s, omerf_scene_info *out)
{
    if (!s || !out) return invalid("null scene/out_info");
    out->device_bytes = s->device_bytes;
    out->pyramid_levels = s->dev.n_levels;
    out->sampler = s->dev.sampler;
    out->occ_bits_set = s->occ_bits_set;
    out->grid_bytes = s->grid_bytes;
    out->grid_blocks_total = s->blocks_total;
    out->grid_blocks_allocated = s->blocks_allocated;
    out->plane_bytes = s->plane_bytes;
    for (int i = 0; i < 2; i++) {
        out->xz_band[i] = s->band[i];
        out->yz_band[i] = s->band[2 + i];
    }
    return OMERF_OK;
}

extern "C" int omerf_scene_get_pyramid_level(const omerf_scene *s, int level, int32_t *nx, int32_t *ny,
                                             float *out_min, float *out_max)
{
    if (!s || !nx || !ny) return invalid("null scene/nx/ny");
    if (level < 0 || level >= s->dev.n_levels) return invalid("pyramid level out of range");
    *nx = s->dev.lvl_nx[level];
    *ny = s->dev.lvl_ny[level];
    if (!out_min && !out_max) return OMERF_OK;
    if (!out_min || !out_max) return invalid("out_min and out_max must both be given");
    size_t n = (size_t)*nx * *ny;
    float2 *tmp = new (std::nothrow) float2[n];
    if (!tmp) {
        omerf_set_error("host allocation failed");
        return OMERF_ERR_NOMEM;
    }
    cudaError_t e = cudaMemcpy(tmp, s->dev.pyr + s->dev.lvl_off[level], n * sizeof(float2), cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) {
        delete[] tmp;
        return omerf_cuda_fail(e, "cudaMemcpy pyramid");
    }
    for (size_t i = 0; i < n; i++) {
        out_min[i] = tmp[i].x;
        out_max[i] = tmp[i].y;
    }
    delete[] tmp;
    return OMERF_OK;
}

extern "C" int omerf_scene_get_block_table(const omerf_scene *s, int32_t *out_table, uint64_t n)
{
    if (!s || !out_table) return invalid("null scene/out_table");
    if (!s->dev.blk_shift) return invalid("scene has no block table (grid_block is 0)");
    if (n != s->blocks_total) return invalid("n does not match grid_blocks_total");
    OMERF_CUDA(cudaMemcpy(out_table, s->d_blk_table, n * sizeof(int32_t), cudaMemcpyDeviceToHost));
    return OMERF_OK;
}

extern "C" int omerf_scene_get_bitfield(const omerf_scene *s, uint32_t *out_words, uint64_t n_words)
{
    if (!s || !out_words) return invalid("null scene/out_words");
    if (s->dev.sampler != OMERF_SAMPLER_GRID) return invalid("scene has no bitfield (sampler is not GRID)");
    uint64_t need = ((uint64_t)s->dev.N[0] * s->dev.N[1] * s->dev.N[2] + 31) / 32;
    if (n_words != need) return invalid("n_words does not match (Nx*Ny*Nz+31)/32");
    OMERF_CUDA(cudaMemcpy(out_words, s->dev.occ, need * 4, cudaMemcpyDeviceToHost));
    return OMERF_OK;
}
