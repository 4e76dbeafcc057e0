// omerf_render.cu — S2..S9 of the hot path: one persistent kernel per frame batch.
//
// Persistent warps with ray refill.  Each lane owns one ray at a time and is in one of four states:
//   IDLE -> (refill: S2 ray generation + S3 box clip) -> TRAV -> READY -> (sample) -> TRAV ... -> FIN -> IDLE
// A warp round runs, in this order and only when enough lanes want it, (1) retire: deferred MLP + store for
// FIN lanes, (2) refill: IDLE lanes take the next pixels of the warp's current 8x4 tile (tiles come from a
// global atomic counter), (3) one traversal step for TRAV lanes, (4) one sample for READY lanes.  Rays have
// very different lengths (about 4 samples on average, a long tail, many sky rays with none), so binding a ray
// to a lane for the whole kernel leaves two thirds of the lanes idle (measured: 10.5 of 32 lanes active);
// refill keeps the expensive phases (sample: ~450 instructions, MLP: ~1100) close to full.
//
//   S2 ray generation          fp32, one correctly rounded operation per step (bit-exact with the CPU checker)
//   S3 box clip                fp32 slab test, padded by 2 lattice indices (the exact per-sample predicate decides)
//   S4 occupancy-plane march   hierarchical DDA over the min/max pyramid of (z_min, z_max): in empty space the
//                              ray jumps to the exit of the coarsest empty node or to the start of the node's
//                              z-interval; every jump is VERIFIED with the exact lattice
//                              arithmetic, so skipping never changes which samples exist
//   S5 gather                  trilinear grid + 3 bilinear planes, uint8 x 8 channels per 8-byte load,
//                              8-bit fixed-point weights, exact integer sums (Eq. 2, R9)
//   S6 activations             exp (exp_q on the decision path), sigmoid (Eq. 3)
//   S7 compositing             front to back, integer optical depth decides termination (Eq. 1/8, R7/R8)
//   S8 deferred MLP            34 -> 16 -> 16 -> 3 in FFMA, weights read from the constant bank (Eq. 4)
//   S9 outputs                 rgb fp32 + per-pixel sample count (Fig. 1)
//
// Why jumps are exact: the lattice point p_k = fma(t_k, d, o) is monotone
// in k in every component (rounding is monotone), so cell indices and z are monotone in k.  If samples k
// and kk both lie in one pyramid node and both are on the same side outside its [min,max] z-range, so
// does every sample between them: all of them fail the predicate and may be skipped.
#include "omerf_device.cuh"

namespace {

enum : int { ST_IDLE = 0, ST_TRAV = 1, ST_READY = 2, ST_FIN = 3 };

// scheduling thresholds (lanes): tuned on B200 with configs[1]
#ifndef OMERF_RETIRE_T
#define OMERF_RETIRE_T 12
#endif
#ifndef OMERF_REFILL_T
#define OMERF_REFILL_T 8
#endif
#ifndef OMERF_SAMPLE_T
#define OMERF_SAMPLE_T 20
#endif

struct Ray {
    float ox, oy, oz, dx, dy, dz;
    float ix, iy, iz; // reciprocals of d (INF where d == 0), proposals only
};

__device__ __forceinline__ float exp_q(float x)
{
    float y = __fmul_rn(x, 0x1.715476p+0f);
    float n = rintf(y);
    float f = __fmaf_rn(n, -0x1.62e4p-1f, x);
    f = __fmaf_rn(n, -0x1.7f7d1cp-20f, f);
    float p = (float)(1.0 / 720.0);
    p = __fmaf_rn(p, f, (float)(1.0 / 120.0));
    p = __fmaf_rn(p, f, (float)(1.0 / 24.0));
    p = __fmaf_rn(p, f, (float)(1.0 / 6.0));
    p = __fmaf_rn(p, f, 0.5f);
    p = __fmaf_rn(p, f, 1.0f);
    p = __fmaf_rn(p, f, 1.0f);
    int e = (int)n + 127;
    e = min(max(e, 1), 254);
    return __fmul_rn(p, __int_as_float(e << 23));
}

__device__ __forceinline__ void lattice_point(const Ray &r, float step, int k, float &px, float &py, float &pz)
{
    float t = __fmul_rn(__fadd_rn(__int2float_rn(k), 0.5f), step);
    px = __fmaf_rn(t, r.dx, r.ox);
    py = __fmaf_rn(t, r.dy, r.oy);
    pz = __fmaf_rn(t, r.dz, r.oz);
}

__device__ __forceinline__ bool in_box(const DevScene &sc, float px, float py, float pz)
{
    return px >= 0.0f && px < sc.box[0] && py >= 0.0f && py < sc.box[1] && pz >= 0.0f && pz < sc.box[2];
}

__device__ __forceinline__ int cell_index(float p, float s, int M)
{
    int i = (int)floorf(__fmaf_rn(p, s, 0.5f));
    return min(max(i, 0), M - 1);
}

__device__ __forceinline__ int voxel_index(float p, float s, int N)
{
    int j = (int)floorf(__fmul_rn(p, s));
    return min(max(j, 0), N - 1);
}

// last lattice index whose parameter is below t_end (proposal only; verified by the caller)
__device__ __forceinline__ int index_before(float t_end, float inv_step, int k1)
{
    float f = ceilf(fmaf(t_end, inv_step, -0.5f)) - 1.0f;
    return f >= (float)k1 ? k1 : (int)f;
}

// ---------------------------------------------------------------------------------- S4: one traversal step
// sampler PLANE.  Advances (k, lvl); returns ST_READY when lattice sample k passes the predicate (Eq. 7),
// ST_FIN when no sample is left, ST_TRAV otherwise.
__device__ __forceinline__ int trav_step_plane(const DevScene &sc, const Ray &r, int &k, int k1, int &lvl)
{
    if (k > k1) return ST_FIN;
    float px, py, pz;
    lattice_point(r, sc.step, k, px, py, pz);
    const int top = sc.n_levels - 1;
    // cell indices are clamped, so points of the 2-index padding outside the box still address valid nodes;
    // the box test is only needed where a sample is declared
    const int ix = cell_index(px, sc.sx, sc.Mx), iy = cell_index(py, sc.sy, sc.My);
    const int nx = ix >> lvl, ny = iy >> lvl;
    const float2 h = __ldg(sc.pyr + sc.lvl_off[lvl] + nx * sc.lvl_ny[lvl] + ny);
    const bool above = pz > h.y, below = pz < h.x;
    if (!above && !below) {
        if (lvl == 0) {
            if (in_box(sc, px, py, pz)) return ST_READY; // z_min <= z <= z_max at the nearest grid point (Eq. 7)
            k++;
            return ST_TRAV;
        }
        lvl--;
        return ST_TRAV;
    }
    // outside the node's z-range: propose a jump to the node's xy exit or to where z reaches the range.
    // The boundary crossed decides the next level: an even boundary index also leaves the parent node.
    const int bxi = nx + (r.dx > 0.0f ? 1 : 0), byi = ny + (r.dy > 0.0f ? 1 : 0);
    const float xb = fmaf((float)(bxi << lvl), sc.cell_x, -0.5f * sc.cell_x);
    const float yb = fmaf((float)(byi << lvl), sc.cell_y, -0.5f * sc.cell_y);
    const float tx = r.dx != 0.0f ? (xb - r.ox) * r.ix : INFINITY;
    const float ty = r.dy != 0.0f ? (yb - r.oy) * r.iy : INFINITY;
    float tz = INFINITY;
    if (above && !below && r.dz < 0.0f) tz = (h.y - r.oz) * r.iz;
    if (below && !above && r.dz > 0.0f) tz = (h.x - r.oz) * r.iz;
    const float t_end = fminf(fminf(tx, ty), tz);
    const int kk = index_before(t_end, sc.inv_step, k1);
    if (kk > k) {
        float qx, qy, qz;
        lattice_point(r, sc.step, kk, qx, qy, qz);
        const int jx = cell_index(qx, sc.sx, sc.Mx) >> lvl, jy = cell_index(qy, sc.sy, sc.My) >> lvl;
        const bool same_side = (above ? qz > h.y : true) && (below ? qz < h.x : true);
        if (jx == nx && jy == ny && same_side) {
            k = kk + 1;
            if (tz <= fminf(tx, ty)) {
                lvl = max(lvl - 1, 0); // entering the node's z-range: refine
            } else {
                const int crossed = tx <= ty ? bxi : byi;
                const int up = crossed == 0 ? 31 : __ffs(crossed) - 1; // levels whose boundary this also is
                lvl = min(lvl + min(up, 2), top);
            }
            return ST_TRAV;
        }
    }
    if (lvl > 0) lvl--;
    else k++; // level 0 and the predicate is false at k
    return ST_TRAV;
}

__device__ __forceinline__ bool occ_test(const DevScene &sc, int lvl, int jx, int jy, int jz)
{
    unsigned long long idx = ((unsigned long long)jx * sc.occ_ny[lvl] + jy) * sc.occ_nz[lvl] + jz;
    return (__ldg(sc.occ + sc.occ_off[lvl] + (idx >> 5)) >> (idx & 31)) & 1u;
}

// sampler GRID (config-4 comparator): multi-resolution binary occupancy grid, DDA-style skipping.
__device__ __forceinline__ int trav_step_grid(const DevScene &sc, const Ray &r, int &k, int k1, int &lvl)
{
    if (k > k1) return ST_FIN;
    float px, py, pz;
    lattice_point(r, sc.step, k, px, py, pz);
    if (!in_box(sc, px, py, pz)) {
        k++;
        return ST_TRAV;
    }
    const int top = sc.occ_levels - 1;
    const int nx = voxel_index(px, sc.ns[0], sc.N[0]) >> lvl, ny = voxel_index(py, sc.ns[1], sc.N[1]) >> lvl,
              nz = voxel_index(pz, sc.ns[2], sc.N[2]) >> lvl;
    if (occ_test(sc, lvl, nx, ny, nz)) {
        if (lvl == 0) return ST_READY;
        lvl--;
        return ST_TRAV;
    }
    const int bxi = nx + (r.dx > 0.0f ? 1 : 0), byi = ny + (r.dy > 0.0f ? 1 : 0), bzi = nz + (r.dz > 0.0f ? 1 : 0);
    const float tx = r.dx != 0.0f ? ((float)(bxi << lvl) * sc.vox[0] - r.ox) * r.ix : INFINITY;
    const float ty = r.dy != 0.0f ? ((float)(byi << lvl) * sc.vox[1] - r.oy) * r.iy : INFINITY;
    const float tz = r.dz != 0.0f ? ((float)(bzi << lvl) * sc.vox[2] - r.oz) * r.iz : INFINITY;
    const float t_end = fminf(fminf(tx, ty), tz);
    const int kk = index_before(t_end, sc.inv_step, k1);
    if (kk > k) {
        float qx, qy, qz;
        lattice_point(r, sc.step, kk, qx, qy, qz);
        if ((voxel_index(qx, sc.ns[0], sc.N[0]) >> lvl) == nx && (voxel_index(qy, sc.ns[1], sc.N[1]) >> lvl) == ny &&
            (voxel_index(qz, sc.ns[2], sc.N[2]) >> lvl) == nz) {
            k = kk + 1;
            const int crossed = (tx <= ty && tx <= tz) ? bxi : (ty <= tz ? byi : bzi);
            const int up = crossed == 0 ? 31 : __ffs(crossed) - 1;
            lvl = min(lvl + min(up, 2), top);
            return ST_TRAV;
        }
    }
    if (lvl > 0) lvl--;
    else k++;
    return ST_TRAV;
}

// ---------------------------------------------------------------------------------- S5: gather (Eq. 2)
__device__ __forceinline__ void axis_tap(float p, float s, int N, int &i0, int &i1, uint32_t &w)
{
    const float q = __fmaf_rn(p, s, -0.5f);
    const int i = __float2int_rd(q);
    // (q - floor q) * 256 is exact, so one fma rounds exactly like the mul followed by the add
    w = (uint32_t)__float2int_rd(__fmaf_rn(__fsub_rn(q, __int2float_rn(i)), 256.0f, 0.5f));
    i0 = min(max(i, 0), N - 1);
    i1 = min(max(i + 1, 0), N - 1);
}

// byte c of x, zero-extended: one PRMT
__device__ __forceinline__ uint32_t byte_of(uint32_t x, int c) { return __byte_perm(x, 0u, 0x4440u + (uint32_t)c); }

// out[c] (+)= sum over the 2x2 footprint of w_ab * texel_ab[c]; exact integers <= 255 * 2^16
template <bool ACCUM>
__device__ __forceinline__ void bilinear8(const uint2 *__restrict__ tex, int Nb, int a0, int a1, uint32_t wa, int b0,
                                          int b1, uint32_t wb, uint32_t out[8])
{
    const uint2 t00 = __ldg(tex + (size_t)a0 * Nb + b0);
    const uint2 t01 = __ldg(tex + (size_t)a0 * Nb + b1);
    const uint2 t10 = __ldg(tex + (size_t)a1 * Nb + b0);
    const uint2 t11 = __ldg(tex + (size_t)a1 * Nb + b1);
    const uint32_t w00 = (256u - wa) * (256u - wb), w10 = wa * (256u - wb), w01 = (256u - wa) * wb, w11 = wa * wb;
#pragma unroll
    for (int c = 0; c < 4; c++) {
        uint32_t lo = w00 * byte_of(t00.x, c) + w10 * byte_of(t10.x, c) + w01 * byte_of(t01.x, c) + w11 * byte_of(t11.x, c);
        uint32_t hi = w00 * byte_of(t00.y, c) + w10 * byte_of(t10.y, c) + w01 * byte_of(t01.y, c) + w11 * byte_of(t11.y, c);
        if (ACCUM) {
            out[c] += lo;
            out[4 + c] += hi;
        } else {
            out[c] = lo;
            out[4 + c] = hi;
        }
    }
}

__device__ __forceinline__ void gather_features(const DevScene &sc, float px, float py, float pz, uint32_t I[8])
{
    int x0, x1, y0, y1, z0, z1;
    uint32_t wx, wy, wz;
    // low-res voxel grid V: bilinear in (x,y) on two z-slices, then the z lerp with rounding (R9)
    axis_tap(px, sc.gs[0], sc.G[0], x0, x1, wx);
    axis_tap(py, sc.gs[1], sc.G[1], y0, y1, wy);
    axis_tap(pz, sc.gs[2], sc.G[2], z0, z1, wz);
    {
        const int Gy = sc.G[1], Gz = sc.G[2];
        const uint2 *g = sc.grid;
        const size_t r00 = ((size_t)x0 * Gy + y0) * Gz, r10 = ((size_t)x1 * Gy + y0) * Gz;
        const size_t r01 = ((size_t)x0 * Gy + y1) * Gz, r11 = ((size_t)x1 * Gy + y1) * Gz;
        const uint2 a00 = __ldg(g + r00 + z0), b00 = __ldg(g + r00 + z1);
        const uint2 a10 = __ldg(g + r10 + z0), b10 = __ldg(g + r10 + z1);
        const uint2 a01 = __ldg(g + r01 + z0), b01 = __ldg(g + r01 + z1);
        const uint2 a11 = __ldg(g + r11 + z0), b11 = __ldg(g + r11 + z1);
        const uint32_t w00 = (256u - wx) * (256u - wy), w10 = wx * (256u - wy), w01 = (256u - wx) * wy, w11 = wx * wy;
#pragma unroll
        for (int c = 0; c < 4; c++) {
            uint32_t A = w00 * byte_of(a00.x, c) + w10 * byte_of(a10.x, c) + w01 * byte_of(a01.x, c) + w11 * byte_of(a11.x, c);
            uint32_t B = w00 * byte_of(b00.x, c) + w10 * byte_of(b10.x, c) + w01 * byte_of(b01.x, c) + w11 * byte_of(b11.x, c);
            I[c] = ((256u - wz) * A + wz * B + 128u) >> 8;
            A = w00 * byte_of(a00.y, c) + w10 * byte_of(a10.y, c) + w01 * byte_of(a01.y, c) + w11 * byte_of(a11.y, c);
            B = w00 * byte_of(b00.y, c) + w10 * byte_of(b10.y, c) + w01 * byte_of(b01.y, c) + w11 * byte_of(b11.y, c);
            I[4 + c] = ((256u - wz) * A + wz * B + 128u) >> 8;
        }
    }
    // triplanes: xy sampled with (x,y), xz with (x,z), yz with (y,z)
    int a0, a1, b0, b1;
    uint32_t wa, wb;
    axis_tap(px, sc.xy_s[0], sc.xy_n[0], a0, a1, wa);
    axis_tap(py, sc.xy_s[1], sc.xy_n[1], b0, b1, wb);
    bilinear8<true>(sc.pxy, sc.xy_n[1], a0, a1, wa, b0, b1, wb, I);
    axis_tap(px, sc.xz_s[0], sc.xz_n[0], a0, a1, wa);
    axis_tap(pz, sc.xz_s[1], sc.xz_n[1], b0, b1, wb);
    bilinear8<true>(sc.pxz, sc.xz_n[1], a0, a1, wa, b0, b1, wb, I);
    axis_tap(py, sc.yz_s[0], sc.yz_n[0], a0, a1, wa);
    axis_tap(pz, sc.yz_s[1], sc.yz_n[1], b0, b1, wb);
    bilinear8<true>(sc.pyz, sc.yz_n[1], a0, a1, wa, b0, b1, wb, I);
}

__device__ __forceinline__ float sigmoid_fast(float x) { return __fdividef(1.0f, 1.0f + __expf(-x)); }

// ---------------------------------------------------------------------------------- S8: deferred MLP (Eq. 4)
__device__ __forceinline__ void deferred_mlp(const DevScene &sc, const float acc[7], const Ray &r, float S[3])
{
    float in[OMERF_MLP_IN];
#pragma unroll
    for (int i = 0; i < 7; i++) in[i] = acc[i];
    const float d[3] = {r.dx, r.dy, r.dz};
#pragma unroll
    for (int c = 0; c < 3; c++) {
        in[7 + c] = d[c];
        float s, co;
        sincosf(d[c], &s, &co); // |d| <= 1: no range reduction slow path
#pragma unroll
        for (int j = 0; j < 4; j++) {
            in[10 + (3 * j + c) * 2] = s;
            in[10 + (3 * j + c) * 2 + 1] = co;
            const float s2 = 2.0f * s * co, c2 = 1.0f - 2.0f * s * s; // double-angle: sin/cos(2^(j+1) d)
            s = s2;
            co = c2;
        }
    }
    float h1[OMERF_MLP_HID], h2[OMERF_MLP_HID];
#pragma unroll
    for (int o = 0; o < OMERF_MLP_HID; o++) {
        float a = sc.b0[o];
#pragma unroll
        for (int i = 0; i < OMERF_MLP_IN; i++) a = fmaf(sc.W0[o * OMERF_MLP_IN + i], in[i], a);
        h1[o] = fmaxf(a, 0.0f);
    }
#pragma unroll
    for (int o = 0; o < OMERF_MLP_HID; o++) {
        float a = sc.b1[o];
#pragma unroll
        for (int i = 0; i < OMERF_MLP_HID; i++) a = fmaf(sc.W1[o * OMERF_MLP_HID + i], h1[i], a);
        h2[o] = fmaxf(a, 0.0f);
    }
#pragma unroll
    for (int o = 0; o < 3; o++) {
        float a = sc.b2[o];
#pragma unroll
        for (int i = 0; i < OMERF_MLP_HID; i++) a = fmaf(sc.W2[o * OMERF_MLP_HID + i], h2[i], a);
        S[o] = sigmoid_fast(a);
    }
}

// ---------------------------------------------------------------------------------- S2 + S3: new ray for a lane
// Returns false when the ray cannot have samples (misses the padded box).
__device__ __forceinline__ bool setup_ray(const DevScene &sc, const omerf_camera &cam, int u, int v, Ray &r, int &k,
                                          int &k1)
{
    // S2 (R19): every step one correctly rounded fp32 operation
    const float a = __fdiv_rn(__fsub_rn(__fadd_rn(__int2float_rn(u), 0.5f), cam.cx), cam.fx);
    const float b = -__fdiv_rn(__fsub_rn(__fadd_rn(__int2float_rn(v), 0.5f), cam.cy), cam.fy);
    const float gx = __fmaf_rn(a, cam.right[0], __fmaf_rn(b, cam.up[0], cam.fwd[0]));
    const float gy = __fmaf_rn(a, cam.right[1], __fmaf_rn(b, cam.up[1], cam.fwd[1]));
    const float gz = __fmaf_rn(a, cam.right[2], __fmaf_rn(b, cam.up[2], cam.fwd[2]));
    const float len2 = __fmaf_rn(gx, gx, __fmaf_rn(gy, gy, __fmul_rn(gz, gz)));
    const float inv = __fdiv_rn(1.0f, __fsqrt_rn(len2));
    r.ox = cam.origin[0];
    r.oy = cam.origin[1];
    r.oz = cam.origin[2];
    r.dx = __fmul_rn(gx, inv);
    r.dy = __fmul_rn(gy, inv);
    r.dz = __fmul_rn(gz, inv);
    r.ix = r.dx != 0.0f ? __fdividef(1.0f, r.dx) : INFINITY; // proposals only: approximate is fine
    r.iy = r.dy != 0.0f ? __fdividef(1.0f, r.dy) : INFINITY;
    r.iz = r.dz != 0.0f ? __fdividef(1.0f, r.dz) : INFINITY;
    // S3: slab test against the box; padded by 2 lattice indices on both sides
    float t0 = 0.0f, t1 = INFINITY;
    bool miss = false;
    const float o[3] = {r.ox, r.oy, r.oz}, d[3] = {r.dx, r.dy, r.dz}, id[3] = {r.ix, r.iy, r.iz};
#pragma unroll
    for (int i = 0; i < 3; i++) {
        if (d[i] == 0.0f) {
            if (o[i] < 0.0f || o[i] > sc.box[i]) miss = true;
        } else {
            const float ta = (0.0f - o[i]) * id[i], tb = (sc.box[i] - o[i]) * id[i];
            t0 = fmaxf(t0, fminf(ta, tb));
            t1 = fminf(t1, fmaxf(ta, tb));
        }
    }
    if (miss || !(t0 <= t1 * 1.0001f + 1e-3f)) return false; // slack far below the 2-index padding
    const float fa = floorf(t0 * sc.inv_step - 0.5f) - 2.0f;
    const float fb = ceilf(t1 * sc.inv_step - 0.5f) + 2.0f;
    k = fa > 0.0f ? (int)fminf(fa, 1.0e9f) : 0;
    k1 = (int)fminf(fb, 1.0e9f);
    return k <= k1;
}

// ---------------------------------------------------------------------------------- the persistent kernel
template <int SAMPLER>
__global__ void __launch_bounds__(128)
omerf_march_kernel(const __grid_constant__ DevScene sc, const omerf_camera *__restrict__ cams, int n_views, int W, int H,
                   float *__restrict__ out_rgb, uint32_t *__restrict__ out_n, unsigned int *__restrict__ tile_counter)
{
    const unsigned FULL = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    const unsigned lt_mask = (1u << lane) - 1u;
    const int tiles_x = (W + 7) >> 3, tiles_y = (H + 3) >> 2;
    const unsigned tiles_per_view = (unsigned)tiles_x * tiles_y;
    const unsigned total_tiles = tiles_per_view * (unsigned)n_views;
    const int start_lvl = (SAMPLER == OMERF_SAMPLER_PLANE ? sc.n_levels : sc.occ_levels) - 1;

    // lane state
    int status = ST_IDLE;
    Ray r;
    int k = 0, k1 = -1, lvl = 0;
    uint32_t Q = 0, n = 0;
    float acc[7];
    size_t pix = 0;
    // warp state
    unsigned tile = 0;
    int tpos = 32;
    bool more = true;

    while (true) {
        unsigned m_fin = __ballot_sync(FULL, status == ST_FIN);
        unsigned m_busy = __ballot_sync(FULL, status == ST_TRAV || status == ST_READY);
        // (1) retire: deferred MLP + outputs for finished rays (S8, S9)
        if (m_fin && (__popc(m_fin) >= OMERF_RETIRE_T || !m_busy)) {
            if (status == ST_FIN) {
                float S[3];
                deferred_mlp(sc, acc, r, S);
                const float T_end = __expf(-(float)Q * (1.0f / 1048576.0f));
                out_rgb[pix * 3 + 0] = __saturatef(acc[0] + S[0] + T_end * sc.bg[0]);
                out_rgb[pix * 3 + 1] = __saturatef(acc[1] + S[1] + T_end * sc.bg[1]);
                out_rgb[pix * 3 + 2] = __saturatef(acc[2] + S[2] + T_end * sc.bg[2]);
                out_n[pix] = n;
                status = ST_IDLE;
            }
        }
        // (2) refill: idle lanes take the next pixels of the current 8x4 tile
        unsigned m_idle = __ballot_sync(FULL, status == ST_IDLE);
        if (more && (__popc(m_idle) >= OMERF_REFILL_T || !m_busy)) {
            while (true) {
                if (tpos >= 32) {
                    unsigned t = 0;
                    if (lane == 0) t = atomicAdd(tile_counter, 1u);
                    tile = __shfl_sync(FULL, t, 0);
                    tpos = 0;
                    if (tile >= total_tiles) {
                        more = false;
                        break;
                    }
                }
                m_idle = __ballot_sync(FULL, status == ST_IDLE);
                if (!m_idle) break;
                const int slot = tpos + __popc(m_idle & lt_mask);
                const bool take = status == ST_IDLE && slot < 32;
                if (take) {
                    const unsigned view = tile / tiles_per_view, tv = tile - view * tiles_per_view;
                    const int ty = (int)(tv / (unsigned)tiles_x), tx = (int)(tv - (unsigned)ty * tiles_x);
                    const int u = tx * 8 + (slot & 7), v = ty * 4 + (slot >> 3);
                    if (u < W && v < H) {
                        const omerf_camera cam = cams[view];
                        pix = ((size_t)view * H + v) * W + u;
                        if (setup_ray(sc, cam, u, v, r, k, k1)) {
                            status = ST_TRAV;
                            lvl = start_lvl;
                            Q = 0;
                            n = 0;
#pragma unroll
                            for (int c = 0; c < 7; c++) acc[c] = 0.0f;
                        } else { // cannot hit the box: background (R14)
                            out_rgb[pix * 3 + 0] = sc.bg[0];
                            out_rgb[pix * 3 + 1] = sc.bg[1];
                            out_rgb[pix * 3 + 2] = sc.bg[2];
                            out_n[pix] = 0;
                        }
                    }
                }
                tpos += min(__popc(m_idle), 32 - tpos);
            }
        }
        if (!__any_sync(FULL, status != ST_IDLE)) {
            if (!more) break;
            continue;
        }
        // (3) one traversal step for rays in empty space / between samples (S4)
        if (status == ST_TRAV) {
            status = SAMPLER == OMERF_SAMPLER_PLANE ? trav_step_plane(sc, r, k, k1, lvl) : trav_step_grid(sc, r, k, k1, lvl);
            if (status == ST_FIN && n == 0) { // no sample at all: background exactly, MLP skipped (R14)
                out_rgb[pix * 3 + 0] = sc.bg[0];
                out_rgb[pix * 3 + 1] = sc.bg[1];
                out_rgb[pix * 3 + 2] = sc.bg[2];
                out_n[pix] = 0;
                status = ST_IDLE;
            }
        }
        // (4) one sample for rays that stand on an occupied lattice point (S5, S6, S7)
        const unsigned m_ready = __ballot_sync(FULL, status == ST_READY);
        const unsigned m_trav = __ballot_sync(FULL, status == ST_TRAV);
        if (m_ready && (__popc(m_ready) >= OMERF_SAMPLE_T || !m_trav)) {
            if (status == ST_READY) {
                float px, py, pz;
                lattice_point(r, sc.step, k, px, py, pz);
                uint32_t I[8];
                gather_features(sc, px, py, pz, I);
                float t[8];
#pragma unroll
                for (int c = 0; c < 8; c++) t[c] = __fmaf_rn(__uint2float_rn(I[c]), sc.deq_mul, sc.deq_add);
                const float tau = exp_q(t[0]); // decision path
                const float od = __fmul_rn(tau, sc.step);
                const uint32_t qk = (uint32_t)rintf(fminf(__fmul_rn(od, 1048576.0f), (float)sc.q_stop));
                const float T = __expf(-(float)Q * (1.0f / 1048576.0f)); // colour path: fast math
                const float wgt = T * (1.0f - __expf(-od));
#pragma unroll
                for (int c = 0; c < 7; c++) acc[c] = fmaf(wgt, sigmoid_fast(t[1 + c]), acc[c]);
                Q += qk;
                n += 1;
                k += 1;
                if (Q >= sc.q_stop) {
                    status = ST_FIN; // early stop (R7)
                } else {
                    // inside the slab the next lattice point is usually occupied too: test it here (level 0)
                    // instead of paying a traversal round for it
                    status = ST_TRAV;
                    lvl = 0;
                    if (SAMPLER == OMERF_SAMPLER_PLANE && k <= k1) {
                        lattice_point(r, sc.step, k, px, py, pz);
                        const int ix = cell_index(px, sc.sx, sc.Mx), iy = cell_index(py, sc.sy, sc.My);
                        const float2 h = __ldg(sc.pyr + ix * sc.My + iy);
                        if (h.x <= pz && pz <= h.y && in_box(sc, px, py, pz)) status = ST_READY;
                    }
                }
            }
        }
    }
}

} // namespace

int omerf_launch_render(const omerf_scene *s, const omerf_camera *d_cams, int n_views, int W, int H, float *out_rgb,
                        uint32_t *out_n, cudaStream_t st, int *launches)
{
    if ((long long)((W + 7) / 8) * ((H + 3) / 4) * n_views > 0x7fffffffll) {
        omerf_set_error("invalid argument: image or batch too large");
        return OMERF_ERR_INVALID;
    }
    OMERF_CUDA(cudaMemsetAsync(s->d_tile_counter, 0, sizeof(unsigned int), st));
    const int grid = s->persistent_blocks;
    if (s->dev.sampler == OMERF_SAMPLER_PLANE)
        omerf_march_kernel<OMERF_SAMPLER_PLANE><<<grid, 128, 0, st>>>(s->dev, d_cams, n_views, W, H, out_rgb, out_n,
                                                                       s->d_tile_counter);
    else
        omerf_march_kernel<OMERF_SAMPLER_GRID><<<grid, 128, 0, st>>>(s->dev, d_cams, n_views, W, H, out_rgb, out_n,
                                                                      s->d_tile_counter);
    *launches = 1;
    OMERF_CUDA(cudaGetLastError());
    return OMERF_OK;
}

// resident blocks of the march kernel on this device: the persistent grid size
int omerf_query_persistent_blocks(int sampler, int *blocks)
{
    int dev = 0, sms = 0, per_sm = 0;
    OMERF_CUDA(cudaGetDevice(&dev));
    OMERF_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    if (sampler == OMERF_SAMPLER_PLANE)
        OMERF_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, omerf_march_kernel<OMERF_SAMPLER_PLANE>, 128, 0));
    else
        OMERF_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, omerf_march_kernel<OMERF_SAMPLER_GRID>, 128, 0));
    *blocks = sms * (per_sm > 0 ? per_sm : 1);
    return OMERF_OK;
}
