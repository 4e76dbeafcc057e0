// omerf_render.cu — S2..S9 of the hot path: one persistent kernel per frame batch.
//
// Each warp owns a pool of OMERF_POOL rays in shared memory; a ray is in one of four states:
//   IDLE -> (refill: S2 ray generation + S3 box clip) -> TRAV -> READY -> (sample) -> TRAV ... -> FIN -> IDLE
// A warp round counts the pool by state, lists the slots of ONE state and runs that phase with (nearly) full warps:
// retire (deferred MLP + stores, full batches of 32), sample, traversal visit, or refill with the next 8x4 pixel tile
// from a global atomic counter.  Inside a traversal visit or a sample phase, lanes whose ray has left the state write
// it back and take the next listed rays, so the warp stays full without a new census.  Rays have very different
// lengths (about 4 samples on average, a long tail, some rays with none), so binding a ray to a lane for the whole
// kernel leaves two thirds of the lanes idle (measured: 10.5 of 32 lanes active; the pool runs at 27).
//
//   S2 ray generation          fp32, one correctly rounded operation per step (bit-exact with the CPU checker)
//   S3 box clip                fp32 slab test padded by 2 lattice indices, then the EXACT range of indices inside the box
//                              (the lattice is monotone: probes + bisection), so the march needs no box test or clamp
//   S4 occupancy-plane march   hierarchical DDA over the min/max pyramid of (z_min, z_max): in empty space the
//                              ray jumps to the exit of the coarsest empty node or to the start of the node's
//                              z-interval; every jump is VERIFIED with the exact lattice
//                              arithmetic, so skipping never changes which samples exist
//   S5 gather                  trilinear grid + 3 bilinear planes as 10 sixteen-byte entries (two adjacent texels of
//                              8 uint8 channels, bytes interleaved per channel), 8-bit fixed-point weights, exact integer
//                              sums as IDP.2A dot products (Eq. 2, R9)
//   S6 activations             exp (exp_q on the decision path), sigmoid through MUFU.TANH (Eq. 3)
//   S7 compositing             front to back, integer optical depth decides termination (Eq. 1/8, R7/R8)
//   S8 deferred MLP            34 -> 16 -> 16 -> 3 as 3xTF32 tensor-core tiles, 16 rays at a time, layer-1 fragments built
//                              in registers from the pool (Eq. 4; omerf_mlp.cuh)
//   S9 outputs                 rgb fp32 + per-pixel sample count (Fig. 1)
// plus the gather calibration of SURVEY 8(d) (sample log + omerf_gather_probe_kernel) and, in the GENERAL
// instantiation, the 8(f) variants (soft occupancy of Eq. 6-8, sparse-block grid).
//
// Why jumps are exact: the lattice point p_k = fma(t_k, d, o) is monotone
// in k in every component (rounding is monotone), so cell indices and z are monotone in k.  If samples k
// and kk both lie in one pyramid node and both are on the same side outside its [min,max] z-range, so
// does every sample between them: all of them fail the predicate and may be skipped.
#include <string.h>

#include <type_traits>

#include "omerf_device.cuh"
#include "omerf_mlp.cuh"

// OMERF_CHECKED build (libomerf_checked.so; paper_2404_09531_b200/build.py: build(checked=True)): every global-memory
// index and every pool slot the render kernels use is range-checked on the device.  A violation sets a bit of
// omerf_check_word (read and cleared by omerf_check_errors) and the access goes to element 0 instead, so the run
// completes and reports.  This is the stand-in for compute-sanitizer memcheck, which is closed on the GPU pool
// (profiles/r02_checked_build.md); the shipped library compiles the checks away.
enum : int { CHK_PYR = 0, CHK_GRID, CHK_PXY, CHK_PXZ, CHK_PYZ, CHK_BLK, CHK_OCC, CHK_VIEW, CHK_PIXEL, CHK_SLOT, CHK_LIST };
#ifdef OMERF_CHECKED
__device__ unsigned int omerf_check_word = 0u;
template <typename T>
__device__ __forceinline__ T chk(T i, unsigned long long n, int code)
{
    if ((unsigned long long)i >= n) {
        atomicOr(&omerf_check_word, 1u << code);
        return (T)0;
    }
    return i;
}
#else
#define chk(i, n, code) (i)
#endif

extern "C" unsigned int omerf_check_errors(void)
{
#ifdef OMERF_CHECKED
    unsigned int w = 0xffffffffu, zero = 0u;
    if (cudaDeviceSynchronize() != cudaSuccess || cudaMemcpyFromSymbol(&w, omerf_check_word, sizeof w) != cudaSuccess) return 0xffffffffu;
    cudaMemcpyToSymbol(omerf_check_word, &zero, sizeof zero);
    return w;
#else
    return 0u;
#endif
}

namespace {

enum : int { ST_IDLE = 0, ST_TRAV = 1, ST_READY = 2, ST_FIN = 3 };

// level policy of the pyramid traversal (speed only: every jump is verified), tuned on B200 with configs[1]
constexpr int OMERF_LVL_START = 6;      // first node size: 2^6 cells
constexpr int OMERF_LVL_ENTER = 2;      // levels to descend when a jump ends where z enters the node's range
constexpr int OMERF_LVL_INSIDE = 2;     // levels to descend when the point is inside the node's z-range
constexpr int OMERF_LVL_FAIL = 2;       // levels to descend when the proposed jump could not be verified
constexpr int OMERF_GRID_LVL_INSIDE = 1; // config-4 comparator (occupancy mip chain): levels to descend in an occupied node
constexpr int OMERF_GRID_LVL_FAIL = 2;   // ... and after a proposal that could not be verified
constexpr int OMERF_LVL_UP = 1;         // levels to ascend after a verified jump across an xy node boundary



struct Ray {
    float ox, oy, oz, dx, dy, dz;
    float ix, iy, iz; // reciprocals of d (INF where d == 0), proposals only
};

__device__ __forceinline__ int floor_int(float x) { return __float2int_rd(x); }
__device__ __forceinline__ int ceil_int(float x) { return __float2int_ru(x); } // saturates: +inf -> INT_MAX

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

// Nearest grid point of P_o (Eq. 7) for a point INSIDE the box (0 <= p < X): p s < M - 1 exactly (s = fl((M-1)/X),
// p <= X (1 - 2^-24)), so the rounded fma lies in [1/2, M - 1/2] and the clamp of R1 to [0, M-1] is the identity.  Every
// lattice index a ray keeps lies inside the box (setup_ray), which is what lets the march drop the clamps and box tests.
__device__ __forceinline__ int cell_index_in_box(float p, float s) { return floor_int(__fmaf_rn(p, s, 0.5f)); }

// last lattice index whose parameter is below t_end (proposal only; verified by the caller)
__device__ __forceinline__ int index_before(float t_end, float inv_step, int k1)
{
    // t_end = +inf saturates to INT_MAX (clamped to k1); anything not above k is rejected by the caller
    return max(min(ceil_int(fmaf(t_end, inv_step, -0.5f)), k1 + 1), 0) - 1;
}

// ---------------------------------------------------------------------------------- S4: one traversal step
// Per-ray constants of the occupancy-plane traversal (proposals only: they set where a jump is tried, never whether it
// is taken).  The exit parameter of the node boundary at level-0 cell index b is
//     t = ((b - 1/2) cell - o) / d = fma((float)b, a, c),   a = cell / d,  c = (-cell / 2 - o) / d   (d = 0: a = 0, c = +inf).
struct PlaneTrav {
    float ax, cx, ay, cy;
    int sx, sy; // 1 if the ray moves towards larger indices, else 0: the boundary a node is left through
};

__device__ __forceinline__ void plane_trav_setup(const DevScene &sc, const Ray &r, PlaneTrav &q)
{
    q.ax = r.dx != 0.0f ? sc.cell_x * r.ix : 0.0f;
    q.cx = r.dx != 0.0f ? (-0.5f * sc.cell_x - r.ox) * r.ix : INFINITY;
    q.ay = r.dy != 0.0f ? sc.cell_y * r.iy : 0.0f;
    q.cy = r.dy != 0.0f ? (-0.5f * sc.cell_y - r.oy) * r.iy : INFINITY;
    q.sx = r.dx > 0.0f ? 1 : 0;
    q.sy = r.dy > 0.0f ? 1 : 0;
}

// sampler PLANE.  One step for a ray in state ST_TRAV (any other status passes through): advances (k, lvl) and returns
// ST_READY when lattice sample k passes the predicate (Eq. 7), ST_FIN when no sample is left, ST_TRAV otherwise.
//   inside the node's [min,max]:  level 0 -> the sample is occupied; level > 0 -> descend
//   outside:  propose a jump to the node's xy exit or to where z reaches the range; if the last index before that
//             (kk) is verified to lie in the same node on the same side, k = kk+1 and the level follows the boundary
//             crossed (entering the z-range: descend OMERF_LVL_ENTER; an xy boundary: ascend OMERF_LVL_UP);
//             otherwise descend OMERF_LVL_FAIL levels, or k+1 at level 0.
// Every index in [k, k1] is inside the box (setup_ray), so cell indices need no clamp and the predicate no box test.
// Written without branches (selects only): the warp does not serialise the inside / jump / descend paths.
__device__ __forceinline__ int trav_step_plane(const DevScene &sc, const Ray &r, const PlaneTrav &q, int &k, int k1, int &lvl,
                                               int status)
{
    const bool run = status == ST_TRAV && k <= k1;
    const float t = __fmul_rn(__fadd_rn(__int2float_rn(k), 0.5f), sc.step);
    const float px = __fmaf_rn(t, r.dx, r.ox), py = __fmaf_rn(t, r.dy, r.oy), pz = __fmaf_rn(t, r.dz, r.oz);
    const int nx = cell_index_in_box(px, sc.sx) >> lvl, ny = cell_index_in_box(py, sc.sy) >> lvl;
    float2 h = make_float2(0.0f, 0.0f);
    if (run) h = __ldg(sc.pyr + chk((uint32_t)(sc.lvl_off[lvl] + nx * sc.lvl_ny[lvl] + ny), sc.n_pyr, CHK_PYR)); // lanes without a ray load nothing
    const bool above = pz > h.y, below = pz < h.x, inside = !(above || below);
    const float tx = fmaf((float)((nx + q.sx) << lvl), q.ax, q.cx);
    const float ty = fmaf((float)((ny + q.sy) << lvl), q.ay, q.cy);
    // where z reaches the side of the range the point is outside of; in the past (or NaN / -inf when dz = 0): never
    const float tzr = ((above ? h.y : h.x) - r.oz) * r.iz;
    const float tz = tzr > t ? tzr : INFINITY;
    const float txy = fminf(tx, ty);
    const int kk = index_before(fminf(txy, tz), sc.inv_step, k1);
    float qx, qy, qz;
    lattice_point(r, sc.step, kk, qx, qy, qz);
    const int jx = cell_index_in_box(qx, sc.sx) >> lvl, jy = cell_index_in_box(qy, sc.sy) >> lvl; // kk in (k, k1] when it counts
    // z is monotone along the ray: both ends above the node's maximum (or both below its minimum) and in the node means
    // every index between them is too.  For an empty node (max < min) "above" alone proves it.
    const bool same_side = above ? qz > h.y : qz < h.x;
    const bool jump = !inside && kk > k && jx == nx && jy == ny && same_side;
    const bool ready = run && inside && lvl == 0;
    // next (k, lvl)
    const int top = sc.n_levels - 1;
    const int lvl_jump = tz <= txy ? max(lvl - OMERF_LVL_ENTER, 0) : min(lvl + OMERF_LVL_UP, top);
    const int lvl_next = inside ? max(lvl - OMERF_LVL_INSIDE, 0) : (jump ? lvl_jump : max(lvl - OMERF_LVL_FAIL, 0));
    const int k_next = jump ? kk + 1 : ((lvl == 0 && !ready) ? k + 1 : k); // level 0 and the predicate is false at k
    if (run) {
        k = k_next;
        lvl = lvl_next;
    }
    return status != ST_TRAV ? status : (k > k1 && !ready ? ST_FIN : (ready ? ST_READY : ST_TRAV));
}

__device__ __forceinline__ bool occ_test(const DevScene &sc, int lvl, int jx, int jy, int jz)
{
    unsigned long long idx = ((unsigned long long)jx * sc.occ_ny[lvl] + jy) * sc.occ_nz[lvl] + jz;
    return (__ldg(sc.occ + chk(sc.occ_off[lvl] + (idx >> 5), sc.n_occ_words, CHK_OCC)) >> (idx & 31)) & 1u;
}

// sampler GRID (config-4 comparator): multi-resolution binary occupancy grid, DDA-style skipping.
// Voxel index of R18 for a point inside the box: floor(p N/X) >= 0; the product can round up to N just below the far
// face, so the upper clamp stays.
__device__ __forceinline__ int voxel_index_in_box(float p, float s, int N) { return min(floor_int(__fmul_rn(p, s)), N - 1); }

// Per-ray constants (proposals only): exit parameter of the voxel boundary at level-0 index b along an axis,
// t = (b vox - o) / d = fma((float)b, vox / d, -o / d)   (d = 0: a = 0, c = +inf).
struct GridTrav {
    float a[3], c[3];
    int s[3];
};

__device__ __forceinline__ void grid_trav_setup(const DevScene &sc, const Ray &r, GridTrav &q)
{
    const float d[3] = {r.dx, r.dy, r.dz}, o[3] = {r.ox, r.oy, r.oz}, id[3] = {r.ix, r.iy, r.iz};
#pragma unroll
    for (int i = 0; i < 3; i++) {
        q.a[i] = d[i] != 0.0f ? sc.vox[i] * id[i] : 0.0f;
        q.c[i] = d[i] != 0.0f ? -o[i] * id[i] : INFINITY;
        q.s[i] = d[i] > 0.0f ? 1 : 0;
    }
}

// Same shape as trav_step_plane: branch-free, a status other than ST_TRAV passes through, every index in [k, k1] is
// inside the box.  An empty node is left through its nearest face (verified: index kk still lies in the node); the level
// then rises as far as the face crossed is aligned.
__device__ __forceinline__ int trav_step_grid(const DevScene &sc, const Ray &r, const GridTrav &q, int &k, int k1, int &lvl, int status)
{
    const bool run = status == ST_TRAV && k <= k1;
    float px, py, pz;
    lattice_point(r, sc.step, k, px, py, pz);
    const int top = sc.occ_levels - 1;
    const int nx = voxel_index_in_box(px, sc.ns[0], sc.N[0]) >> lvl, ny = voxel_index_in_box(py, sc.ns[1], sc.N[1]) >> lvl,
              nz = voxel_index_in_box(pz, sc.ns[2], sc.N[2]) >> lvl;
    bool occ = false;
    if (run) occ = occ_test(sc, lvl, nx, ny, nz); // lanes without a ray load nothing
    const int bxi = nx + q.s[0], byi = ny + q.s[1], bzi = nz + q.s[2];
    const float tx = fmaf((float)(bxi << lvl), q.a[0], q.c[0]);
    const float ty = fmaf((float)(byi << lvl), q.a[1], q.c[1]);
    const float tz = fmaf((float)(bzi << lvl), q.a[2], q.c[2]);
    const int kk = index_before(fminf(fminf(tx, ty), tz), sc.inv_step, k1);
    float qx, qy, qz;
    lattice_point(r, sc.step, kk, qx, qy, qz);
    const bool same = (voxel_index_in_box(qx, sc.ns[0], sc.N[0]) >> lvl) == nx && (voxel_index_in_box(qy, sc.ns[1], sc.N[1]) >> lvl) == ny &&
                      (voxel_index_in_box(qz, sc.ns[2], sc.N[2]) >> lvl) == nz;
    const bool jump = !occ && kk > k && same;
    const bool ready = run && occ && lvl == 0;
    const int crossed = (tx <= ty && tx <= tz) ? bxi : (ty <= tz ? byi : bzi);
    const int up = crossed == 0 ? 2 : min(__ffs(crossed) - 1, 2); // leaving 2^up-aligned parents: ascend that far
    const int lvl_next = occ ? max(lvl - OMERF_GRID_LVL_INSIDE, 0) : (jump ? min(lvl + up, top) : max(lvl - OMERF_GRID_LVL_FAIL, 0));
    const int k_next = jump ? kk + 1 : ((lvl == 0 && !ready) ? k + 1 : k);
    if (run) {
        k = k_next;
        lvl = lvl_next;
    }
    return status != ST_TRAV ? status : (k > k1 && !ready ? ST_FIN : (ready ? ST_READY : ST_TRAV));
}

// ---------------------------------------------------------------------------------- S5: gather (Eq. 2)
// One axis of a bilinear footprint (R9/R10): texel coordinate q = p N/X - 1/2, lower texel floor(q), 8-bit weight
// floor(frac * 256 + 1/2) in [0,256].  Both come out of ONE conversion: F = floor(fma(q, 256, 1/2)) = 256 floor(q) + w
// exactly (256 q is exact and, for q < 2^15, so is the sum up to a rounding that cannot cross an integer), so
// i = F >> 8 and w = F & 255.  A weight of 256 appears as (i + 1, 0): the same texels with the same total weights.
// The point is inside the box (checked before every sample), hence -1 <= i <= N-1; i = -1 (both taps are texel 0) is
// folded into (i, w) = (0, 0), which gives texel 0 the whole weight as well.
__device__ __forceinline__ void axis_tap(float p, float s, int &i, uint32_t &w)
{
    const float q = __fmaf_rn(p, s, -0.5f);
    const int F = max(floor_int(__fmaf_rn(q, 256.0f, 0.5f)), 0);
    i = F >> 8;
    w = (uint32_t)(F & 255);
}

// Bilinear footprints as 16-bit x 8-bit dot products (IDP.2A, fma pipe, full rate): the four weights
// w_ab = (256 - w_a | w_a)(256 - w_b | w_b) are packed as two u16 pairs (pairs along axis b), and an S0 entry already holds
// the bytes of texels b0 and b1 side by side per channel (pair_entry), so a channel costs one IDP.2A per row and no byte
// shuffle.  Only w_00 can reach 2^16 (w_a = w_b = 0; the taps never carry a weight of 256, see axis_tap): it is then
// stored as 65535 and the missing unit of texel (a0, b0) is added (`ovf`, a rare branch): the sum stays the exact integer of R9.
struct BiW {
    uint32_t w0, w1; // (w00 | w01 << 16), (w10 | w11 << 16): pairs along axis b for rows a0 and a1
    bool ovf;
};

__device__ __forceinline__ BiW bilinear_weights(uint32_t wa, uint32_t wb)
{
    // (256 - wb | wb << 16) times a row weight <= 256 gives both products of the row in one multiply
    const uint32_t pb = wb * 0xffffu + 256u;
    BiW r;
    r.ovf = (wa | wb) == 0u;
    r.w0 = r.ovf ? 0xffffu : (256u - wa) * pb;
    r.w1 = wa * pb;
    return r;
}

// acc[0..7] += sum over the 2x2 footprint of w_ab * texel_ab[c]; e0 = entry of row a0 (texels b0, b1), e1 = of row a1
__device__ __forceinline__ void bilinear8_dp(const uint4 e0, const uint4 e1, const BiW w, uint32_t acc[8])
{
    acc[0] = __dp2a_lo(w.w1, e1.x, __dp2a_lo(w.w0, e0.x, acc[0]));
    acc[1] = __dp2a_hi(w.w1, e1.x, __dp2a_hi(w.w0, e0.x, acc[1]));
    acc[2] = __dp2a_lo(w.w1, e1.y, __dp2a_lo(w.w0, e0.y, acc[2]));
    acc[3] = __dp2a_hi(w.w1, e1.y, __dp2a_hi(w.w0, e0.y, acc[3]));
    acc[4] = __dp2a_lo(w.w1, e1.z, __dp2a_lo(w.w0, e0.z, acc[4]));
    acc[5] = __dp2a_hi(w.w1, e1.z, __dp2a_hi(w.w0, e0.z, acc[5]));
    acc[6] = __dp2a_lo(w.w1, e1.w, __dp2a_lo(w.w0, e0.w, acc[6]));
    acc[7] = __dp2a_hi(w.w1, e1.w, __dp2a_hi(w.w0, e0.w, acc[7]));
    if (w.ovf) { // w_00 = 2^16 was stored as 2^16 - 1 (probability 2^-16 per footprint): one more unit of texel (a0, b0)
        acc[0] += e0.x & 255u; acc[1] += (e0.x >> 16) & 255u; acc[2] += e0.y & 255u; acc[3] += (e0.y >> 16) & 255u;
        acc[4] += e0.z & 255u; acc[5] += (e0.z >> 16) & 255u; acc[6] += e0.w & 255u; acc[7] += (e0.w >> 16) & 255u;
    }
}

// Entry indices of the four (x, z) corners of V at tap y, order x0z0, x0z1, x1z0, x1z1; every entry holds the texels
// (y, y+1) of its (x, z) (S0 layout, omerf_build.cu).  Dense layout: row-major [Gx][Gy][Gz]; sparse blocks (8(f).1):
// one block-table lookup per corner, then the entry inside the atlas block (the y+1 texel of an entry was copied from the
// neighbouring block at bake time, so one lookup serves both y taps).
template <bool GENERAL>
__device__ __forceinline__ void grid_corner_offsets(const DevScene &sc, int x0, int x1, int y, int z0, int z1, uint32_t off[4])
{
    if (!GENERAL || sc.blk_shift == 0) {
        const uint32_t Gy = (uint32_t)sc.G[1], Gz = (uint32_t)sc.G[2];
        const uint32_t c0 = ((uint32_t)x0 * Gy + (uint32_t)y) * Gz, c1 = ((uint32_t)x1 * Gy + (uint32_t)y) * Gz;
        off[0] = c0 + (uint32_t)z0;
        off[1] = c0 + (uint32_t)z1;
        off[2] = c1 + (uint32_t)z0;
        off[3] = c1 + (uint32_t)z1;
    } else {
        const int s = sc.blk_shift, m = (1 << s) - 1;
        const int xs[2] = {x0, x1}, zs[2] = {z0, z1};
#pragma unroll
        for (int a = 0; a < 2; a++)
#pragma unroll
            for (int b = 0; b < 2; b++) {
                // every corner of a sample inside the slab lies in an allocated block (R24); max() only guards memory
                const int id = max(__ldg(sc.blk_table + chk((uint32_t)(((xs[a] >> s) * sc.nby + (y >> s)) * sc.nbz + (zs[b] >> s)), sc.n_blk, CHK_BLK)), 0);
                off[a * 2 + b] = ((uint32_t)id << (3 * s)) + (uint32_t)(((((xs[a] & m) << s) + (y & m)) << s) + (zs[b] & m));
            }
    }
}

// The 10 gathers of one sample: every load fetches a PAIR of texels adjacent along y (V) or the second axis (planes) as
// one 16-byte entry.
struct Footprints {
    uint4 g[4];  // V: corners x0z0, x0z1, x1z0, x1z1, each (y0 | y1)
    uint4 p[6];  // xy rows a0, a1; xz rows a0, a1; yz rows a0, a1, each (b0 | b1)
};

template <bool GENERAL>
__device__ __forceinline__ void gather_features(const DevScene &sc, float px, float py, float pz, uint32_t I[8])
{
    // taps and weights of all four sources first, then all 10 loads, then the arithmetic
    int x0, y0, z0;
    uint32_t wx, wy, wz;
    axis_tap(px, sc.gs[0], x0, wx);
    axis_tap(py, sc.gs[1], y0, wy);
    axis_tap(pz, sc.gs[2], z0, wz);
    const int x1 = min(x0 + 1, sc.G[0] - 1), z1 = min(z0 + 1, sc.G[2] - 1);
    Footprints f;
    {
        uint32_t off[4];
        grid_corner_offsets<GENERAL>(sc, x0, x1, y0, z0, z1, off);
#pragma unroll
        for (int c = 0; c < 4; c++) f.g[c] = __ldg(sc.grid + chk(off[c], sc.n_grid, CHK_GRID));
    }
    // triplanes: xy sampled with (x,y), xz with (x,z), yz with (y,z).  When the planes share their resolution per
    // world axis (every config: xy A x A, xz and yz A x B) a tap computed for one plane is the other plane's tap too
    // (same scale, same arithmetic), so three taps serve all six plane axes.
    int xa, ya, za;
    uint32_t xw, yw, zw;
    axis_tap(px, sc.xy_s[0], xa, xw);
    axis_tap(py, sc.xy_s[1], ya, yw);
    axis_tap(pz, sc.xz_s[1], za, zw);
    int xb = xa, yb = ya, zb = za; // taps of xz axis 0, yz axis 0, yz axis 1
    uint32_t xbw = xw, ybw = yw, zbw = zw;
    if (!sc.shared_taps) {
        axis_tap(px, sc.xz_s[0], xb, xbw);
        axis_tap(py, sc.yz_s[0], yb, ybw);
        axis_tap(pz, sc.yz_s[1], zb, zbw);
    }
    {
        // 32-bit entry indices (every source has fewer than 2^32 texels; checked at scene creation)
        const uint32_t Nxy = (uint32_t)sc.xy_n[1], Nxz = (uint32_t)sc.xz_rows, Nyz = (uint32_t)sc.yz_rows;
        const uint32_t xa1 = (uint32_t)min(xa + 1, sc.xy_n[0] - 1), xb1 = (uint32_t)min(xb + 1, sc.xz_n[0] - 1),
                       yb1 = (uint32_t)min(yb + 1, sc.yz_n[0] - 1);
        const uint32_t zr = (uint32_t)(za - sc.xz_zoff), zs = (uint32_t)(zb - sc.yz_zoff); // low-z bake: rows below the band are not stored
        f.p[0] = __ldg(sc.pxy + chk((uint32_t)xa * Nxy + (uint32_t)ya, sc.n_pxy, CHK_PXY));
        f.p[1] = __ldg(sc.pxy + chk(xa1 * Nxy + (uint32_t)ya, sc.n_pxy, CHK_PXY));
        f.p[2] = __ldg(sc.pxz + chk((uint32_t)xb * Nxz + zr, sc.n_pxz, CHK_PXZ));
        f.p[3] = __ldg(sc.pxz + chk(xb1 * Nxz + zr, sc.n_pxz, CHK_PXZ));
        f.p[4] = __ldg(sc.pyz + chk((uint32_t)yb * Nyz + zs, sc.n_pyz, CHK_PYZ));
        f.p[5] = __ldg(sc.pyz + chk(yb1 * Nyz + zs, sc.n_pyz, CHK_PYZ));
    }
    const BiW wg = bilinear_weights(wx, wy);
    const BiW w1 = bilinear_weights(xw, yw), w2 = bilinear_weights(xbw, zw), w3 = bilinear_weights(ybw, zbw);

    uint32_t A[8], B[8];
#pragma unroll
    for (int c = 0; c < 8; c++) A[c] = B[c] = 0u;
    // V: bilinear in (x,y) on the z-slices z0 (entries x0z0, x1z0) and z1 (x0z1, x1z1)
    bilinear8_dp(f.g[0], f.g[2], wg, A);
    bilinear8_dp(f.g[1], f.g[3], wg, B);
    // the z lerp rounds once (R9): (256 - wz) A + wz B < 2^32
#pragma unroll
    for (int c = 0; c < 8; c++) I[c] = ((256u - wz) * A[c] + wz * B[c] + 128u) >> 8;
    bilinear8_dp(f.p[0], f.p[1], w1, I);
    bilinear8_dp(f.p[2], f.p[3], w2, I);
    bilinear8_dp(f.p[4], f.p[5], w3, I);
}

// per-sample activations (Eq. 3, colour path only): sigmoid(2x) = 1/2 + 1/2 tanh(x) with one MUFU.TANH; the caller
// passes HALF the pre-activation (the factor is folded into the dequantisation constants).
// tanh.approx has an absolute error of about 2^-11 = 5e-4, so the sigmoid is off by <= 2.5e-4; the compositing
// weights sum to <= 1, which bounds the contribution to the pixel at 2.5e-4 of the 2e-3 budget.
__device__ __forceinline__ float sigmoid_of_half(float x)
{
    float t;
    asm("tanh.approx.f32 %0, %1;" : "=f"(t) : "f"(x));
    return fmaf(t, 0.5f, 0.5f);
}

// ---------------------------------------------------------------------------------- S2 + S3: new ray for a lane
// S2 (R19): every step one correctly rounded fp32 operation
__device__ __forceinline__ void ray_direction(const omerf_camera &cam, int u, int v, float &dx, float &dy, float &dz)
{
    const float a = __fdiv_rn(__fsub_rn(__fadd_rn(__int2float_rn(u), 0.5f), cam.cx), cam.fx);
    const float b = -__fdiv_rn(__fsub_rn(__fadd_rn(__int2float_rn(v), 0.5f), cam.cy), cam.fy);
    const float gx = __fmaf_rn(a, cam.right[0], __fmaf_rn(b, cam.up[0], cam.fwd[0]));
    const float gy = __fmaf_rn(a, cam.right[1], __fmaf_rn(b, cam.up[1], cam.fwd[1]));
    const float gz = __fmaf_rn(a, cam.right[2], __fmaf_rn(b, cam.up[2], cam.fwd[2]));
    const float len2 = __fmaf_rn(gx, gx, __fmaf_rn(gy, gy, __fmul_rn(gz, gz)));
    const float inv = __fdiv_rn(1.0f, __fsqrt_rn(len2));
    dx = __fmul_rn(gx, inv);
    dy = __fmul_rn(gy, inv);
    dz = __fmul_rn(gz, inv);
}

// Returns false when the ray cannot have samples (misses the padded box).
__device__ __forceinline__ bool setup_ray(const DevScene &sc, const omerf_camera &cam, int u, int v, Ray &r, int &k,
                                          int &k1)
{
    ray_direction(cam, u, v, r.dx, r.dy, r.dz);
    r.ox = cam.origin[0];
    r.oy = cam.origin[1];
    r.oz = cam.origin[2];
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
    if (k > k1) return false;
    // The exact index range inside the box.  Every component of the lattice point is monotone in the index (rounding is
    // monotone), so "entered the box" (per axis: past the face the ray comes in through) is false..false true..true and
    // "not yet left" is true..true false..false: the indices inside the box are [first entered, last not yet left].
    // A few linear probes (the padding is 2 indices), then bisection (rays that graze a face).
    auto entered = [&](int i) {
        float px, py, pz;
        lattice_point(r, sc.step, i, px, py, pz);
        return (r.dx >= 0.0f ? px >= 0.0f : px < sc.box[0]) && (r.dy >= 0.0f ? py >= 0.0f : py < sc.box[1]) &&
               (r.dz >= 0.0f ? pz >= 0.0f : pz < sc.box[2]);
    };
    auto not_left = [&](int i) {
        float px, py, pz;
        lattice_point(r, sc.step, i, px, py, pz);
        return (r.dx >= 0.0f ? px < sc.box[0] : px >= 0.0f) && (r.dy >= 0.0f ? py < sc.box[1] : py >= 0.0f) &&
               (r.dz >= 0.0f ? pz < sc.box[2] : pz >= 0.0f);
    };
    // smallest index in [lo, hi] for which a monotone (false..false true..true) predicate holds, hi + 1 if none: probes
    // next to the estimate first (it is usually right or off by one), then bisection (rays that graze a face)
    auto first_true = [&](auto pred, int lo, int hi, int guess) {
        int L = lo, H = hi + 1, p = min(max(guess, lo), hi);
#pragma unroll 1
        for (int it = 0; L < H; it++) {
            const bool t = pred(p);
            if (t) H = p;
            else L = p + 1;
            p = it < 3 ? (t ? p - 1 : p + 1) : L + ((H - 1 - L) >> 1);
            p = min(max(p, L), max(H - 1, L));
        }
        return L;
    };
    const int ge = (int)fminf(ceilf(t0 * sc.inv_step - 0.5f), 1.0e9f), gl = (int)fminf(floorf(t1 * sc.inv_step - 0.5f), 1.0e9f) + 1;
    const int ka = first_true(entered, k, k1, ge);                                     // first index past the entry faces
    if (ka > k1) return false;
    const int kb = first_true([&](int i) { return !not_left(i); }, ka, k1, gl) - 1;     // last index before the exit faces
    k = ka;
    k1 = kb;
    return k <= k1;
}

// ---------------------------------------------------------------------------------- the persistent kernel
// Warp-private ray pool in shared memory (structure of arrays, one word per ray and field).
constexpr int OMERF_POOL = 96;          // rays per warp; a multiple of 32
constexpr int OMERF_TRAV_STEPS = 48;    // cap on the traversal steps of one visit
constexpr int OMERF_TRAV_KEEP = 16;
constexpr int OMERF_DRAIN_TRAV_KEEP = 1;  // in the endgame and the drain a traversal visit runs until every listed ray is done
constexpr int OMERF_SAMPLE_SWAP = 8;    // lanes that must have left the READY state before they take the next listed rays
constexpr int OMERF_TRAV_SWAP = 8;      // lanes that must be free before they take the next listed rays
constexpr int OMERF_SAMPLE_KEEP = 24;   // sample again at once while this many lanes stand on an occupied point
#define OMERF_WARPS 4
static_assert(OMERF_POOL <= 255, "the census packs the state counts into bytes");
static_assert(OMERF_SAMPLE_SWAP >= 1 && OMERF_SAMPLE_SWAP <= 32 && OMERF_TRAV_SWAP >= 1 && OMERF_TRAV_SWAP <= 32,
              "a swap threshold above the warp size would never release a finished lane");
constexpr int OMERF_ENDGAME_WARPS = 2;   // endgame starts when fewer than this many tiles per warp are left
constexpr int OMERF_ENDGAME_BUSY = 32;   // in the endgame a warp takes a new tile only with at most this many rays in flight
#define OMERF_PJ (OMERF_POOL / 32)

// Entry OMERF_NO_RAY of every per-ray array is the slot of a lane that holds no ray: written once at kernel start
// (an idle ray of view 0 with direction 0 and an empty index range), never listed, never written again.  A lane that
// takes no ray in a swap step loads from it, so it reads nothing another lane may be writing back in the same step.
#define OMERF_NO_RAY OMERF_POOL
struct WarpPool {
    uint32_t meta[OMERF_POOL + 1]; // status (bits 0-1) | pyramid level (bits 2-6) | view (bits 8-31)
    float d[3][OMERF_POOL + 1];    // ray direction
    int k[OMERF_POOL + 1], k1[OMERF_POOL + 1];
    uint32_t Q[OMERF_POOL + 1], n[OMERF_POOL + 1], pix[OMERF_POOL + 1];
    float acc[7][OMERF_POOL + 1];
    uint8_t list[OMERF_POOL]; // slots in the picked state, in slot order (phases other than traversal use the first 32)
};

__device__ __forceinline__ uint32_t pack_meta(int status, int lvl, uint32_t view)
{
    return (uint32_t)status | ((uint32_t)lvl << 2) | (view << 8);
}

// ---------------------------------------------------------------------------------- S4: one traversal visit
// Steps the hierarchical DDA for the rays listed in P.list[0 .. n_sel) (all rays of the pool in state ST_TRAV).  The
// first 32 start at once; when OMERF_TRAV_SWAP lanes have finished their ray (it reached a sample or ran out), those
// lanes write it back and take the next listed rays, so the warp stays full without a new census of the pool.  The
// visit ends when the list is exhausted and fewer than OMERF_TRAV_KEEP lanes still traverse, or after
// OMERF_TRAV_STEPS steps (occupied rays then get their samples).
// per-lane cache of the camera origin of the view last used (rays of one lane almost always share the view)
struct LaunchBounds { // what the OMERF_CHECKED build checks views and pixels against
    uint32_t n_views;
    unsigned long long n_pix;
};
struct OriginCache {
    uint32_t view;
    float ox, oy, oz;
};
__device__ __forceinline__ void ray_origin(OriginCache &oc, const omerf_camera *__restrict__ cams, const LaunchBounds &lb, uint32_t view, Ray &r)
{
    if (view != oc.view) {
        oc.view = view;
        const omerf_camera *cam = cams + chk(view, lb.n_views, CHK_VIEW);
        oc.ox = __ldg(&cam->origin[0]);
        oc.oy = __ldg(&cam->origin[1]);
        oc.oz = __ldg(&cam->origin[2]);
    }
    r.ox = oc.ox;
    r.oy = oc.oy;
    r.oz = oc.oz;
}

struct NoTrav {};
template <int SAMPLER>
struct TravLane {
    Ray r;
    typename std::conditional<SAMPLER == OMERF_SAMPLER_PLANE, PlaneTrav, NoTrav>::type q;
    typename std::conditional<SAMPLER == OMERF_SAMPLER_PLANE, NoTrav, GridTrav>::type g;
    int k, k1, lvl, status, slot; // slot < 0: the lane holds no ray
    uint32_t view;
};

__device__ __forceinline__ void plane_trav_setup(const DevScene &, const Ray &, NoTrav &) {}
__device__ __forceinline__ void grid_trav_setup(const DevScene &, const Ray &, NoTrav &) {}

template <int SAMPLER>
__device__ __forceinline__ void trav_load(const DevScene &sc, const WarpPool &P, const omerf_camera *__restrict__ cams,
                                          const LaunchBounds &lb, OriginCache &oc, int slot, TravLane<SAMPLER> &L)
{
    L.slot = slot;
    const int s_ = slot < 0 ? OMERF_NO_RAY : chk(slot, OMERF_POOL, CHK_SLOT); // lanes without a ray read the constant slot and step nothing
    const uint32_t m = P.meta[s_];
    L.status = slot < 0 ? ST_IDLE : ST_TRAV;
    L.lvl = (int)((m >> 2) & 31u);
    L.view = m >> 8;
    L.k = P.k[s_];
    L.k1 = P.k1[s_];
    L.r.dx = P.d[0][s_];
    L.r.dy = P.d[1][s_];
    L.r.dz = P.d[2][s_];
    ray_origin(oc, cams, lb, L.view, L.r);
    L.r.ix = L.r.dx != 0.0f ? __fdividef(1.0f, L.r.dx) : INFINITY;
    L.r.iy = L.r.dy != 0.0f ? __fdividef(1.0f, L.r.dy) : INFINITY;
    L.r.iz = L.r.dz != 0.0f ? __fdividef(1.0f, L.r.dz) : INFINITY;
    plane_trav_setup(sc, L.r, L.q);
    grid_trav_setup(sc, L.r, L.g);
}

template <int SAMPLER>
__device__ __forceinline__ void trav_store(const DevScene &sc, WarpPool &P, const LaunchBounds &lb, const TravLane<SAMPLER> &L,
                                           float *__restrict__ out_rgb, uint32_t *__restrict__ out_n)
{
    const int s_ = chk(L.slot, OMERF_POOL, CHK_SLOT);
    int st_ = L.status;
    if (st_ == ST_FIN && P.n[s_] == 0) { // no sample at all: background exactly, MLP skipped (R14)
        const size_t pix = chk((size_t)P.pix[s_], lb.n_pix, CHK_PIXEL);
        out_rgb[pix * 3 + 0] = sc.bg[0];
        out_rgb[pix * 3 + 1] = sc.bg[1];
        out_rgb[pix * 3 + 2] = sc.bg[2];
        out_n[pix] = 0;
        st_ = ST_IDLE;
    }
    P.k[s_] = L.k;
    P.meta[s_] = pack_meta(st_, L.lvl, L.view);
}

template <int SAMPLER>
__device__ __forceinline__ void trav_visit(const DevScene &sc, WarpPool &P, const omerf_camera *__restrict__ cams, const LaunchBounds &lb,
                                           OriginCache &oc, int lane, int n_sel, int keep, float *__restrict__ out_rgb, uint32_t *__restrict__ out_n)
{
    const unsigned FULL = 0xffffffffu;
    const unsigned lt_mask = (1u << lane) - 1u;
    TravLane<SAMPLER> L;
    trav_load(sc, P, cams, lb, oc, lane < n_sel ? (int)P.list[lane] : -1, L);
    int next = min(n_sel, 32); // first list entry not yet taken
#pragma unroll 1
    for (int it = 0; it < OMERF_TRAV_STEPS; it++) {
        if constexpr (SAMPLER == OMERF_SAMPLER_PLANE) {
            L.status = trav_step_plane(sc, L.r, L.q, L.k, L.k1, L.lvl, L.status);
        } else {
            L.status = trav_step_grid(sc, L.r, L.g, L.k, L.k1, L.lvl, L.status);
        }
        const unsigned going = __ballot_sync(FULL, L.status == ST_TRAV);
        if (next < n_sel) {
            // lanes whose ray is done (or that hold none) take the next listed rays, a batch at a time
            const bool free_lane = L.status != ST_TRAV;
            const unsigned fm = ~going;
            if (__popc(fm) >= OMERF_TRAV_SWAP) {
                if (free_lane) {
                    if (L.slot >= 0) trav_store(sc, P, lb, L, out_rgb, out_n);
                    const int idx = next + __popc(fm & lt_mask);
                    trav_load(sc, P, cams, lb, oc, idx < n_sel ? (int)P.list[idx] : -1, L);
                }
                next = min(next + __popc(fm), n_sel);
            }
        } else if (__popc(going) < keep) {
            break;
        }
    }
    if (L.slot >= 0) trav_store(sc, P, lb, L, out_rgb, out_n);
}

constexpr int OMERF_MIN_BLOCKS = 5;
// LOG (gather calibration only): every sample taken is appended to sample_log as (pixel, lattice index).
// GENERAL: the 8(f) variants (soft occupancy, sparse-block grid) behind warp-uniform branches; the plain path
// (dense grid, binary mask) is compiled without them.
template <int SAMPLER, bool LOG, bool GENERAL>
__global__ void __launch_bounds__(32 * OMERF_WARPS, OMERF_MIN_BLOCKS)
omerf_march_kernel(const __grid_constant__ DevScene sc, const omerf_camera *__restrict__ cams, int n_views, int W, int H,
                   float *__restrict__ out_rgb, uint32_t *__restrict__ out_n, unsigned int *__restrict__ tile_counter,
                   uint2 *__restrict__ sample_log, unsigned int log_capacity, unsigned int tile_first, unsigned int tile_end)
{
    __shared__ WarpPool pools[OMERF_WARPS];
    WarpPool &P = pools[threadIdx.x >> 5];
    const unsigned FULL = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    const unsigned lt_mask = (1u << lane) - 1u;
    const int tiles_x = (W + 7) >> 3, tiles_y = (H + 3) >> 2;
    const unsigned tiles_per_view = (unsigned)tiles_x * tiles_y;
    const unsigned total_tiles = tile_end; // this launch renders the tiles [tile_first, tile_end) of the batch
    const int start_lvl = min((SAMPLER == OMERF_SAMPLER_PLANE ? sc.n_levels : sc.occ_levels) - 1, OMERF_LVL_START);

#pragma unroll
    for (int j = 0; j < OMERF_PJ; j++) P.meta[lane + 32 * j] = ST_IDLE;
    if (lane == 0) {
        P.meta[OMERF_NO_RAY] = pack_meta(ST_IDLE, 0, 0u);
        P.k[OMERF_NO_RAY] = 0;
        P.k1[OMERF_NO_RAY] = -1;
        P.Q[OMERF_NO_RAY] = P.n[OMERF_NO_RAY] = P.pix[OMERF_NO_RAY] = 0u;
#pragma unroll
        for (int c = 0; c < 3; c++) P.d[c][OMERF_NO_RAY] = 0.0f;
#pragma unroll
        for (int c = 0; c < 7; c++) P.acc[c][OMERF_NO_RAY] = 0.0f;
    }
    __syncwarp();
    bool more = true;
    const LaunchBounds lb = {(uint32_t)n_views, (unsigned long long)n_views * (unsigned long long)W * (unsigned long long)H};
    OriginCache oc = {0xffffffffu, 0.0f, 0.0f, 0.0f};
    // Endgame: a warp's pool holds about three tiles of work, which would all drain at falling utilisation once the
    // tile counter runs out.  For the last tiles, warps refill only when (nearly) empty, so the remaining work
    // spreads over all warps and they finish together.
    bool endgame = false;
    const unsigned endgame_tiles = OMERF_ENDGAME_WARPS * gridDim.x * OMERF_WARPS;

    while (true) {
        // ---- census of the pool: every lane adds 1 << (8 * state) for its slots, one warp reduction (REDUX) gives the four
        // counts as the bytes of one word (a pool holds at most 255 rays); ballots are taken for the picked state only
        uint32_t st_lane[OMERF_PJ], packed = 0;
#pragma unroll
        for (int j = 0; j < OMERF_PJ; j++) {
            st_lane[j] = P.meta[lane + 32 * j] & 3u;
            packed += 1u << (8 * st_lane[j]);
        }
        packed = __reduce_add_sync(FULL, packed);
        const int cnt[4] = {(int)(packed & 255u), (int)((packed >> 8) & 255u), (int)((packed >> 16) & 255u), (int)(packed >> 24)};
        // ---- pick a phase: full warps first, then the fullest (all warp-uniform)
        int phase, n_sel;
        unsigned b[OMERF_PJ];
#define OMERF_PICK(S)                                           \
    {                                                           \
        phase = (S);                                            \
        n_sel = cnt[S];                                         \
    }
        if (cnt[ST_FIN] >= 32) OMERF_PICK(ST_FIN)
        else if (cnt[ST_READY] >= 32) OMERF_PICK(ST_READY)
        else if (cnt[ST_TRAV] >= 32) OMERF_PICK(ST_TRAV)
        else if (more && cnt[ST_IDLE] >= (endgame ? OMERF_POOL - OMERF_ENDGAME_BUSY : 32)) OMERF_PICK(ST_IDLE)
        else if (cnt[ST_READY] > 0 && cnt[ST_READY] >= cnt[ST_TRAV]) OMERF_PICK(ST_READY)
        else if (cnt[ST_TRAV] > 0) OMERF_PICK(ST_TRAV)
        else if (cnt[ST_FIN] > 0) OMERF_PICK(ST_FIN) // finished rays wait for a full MLP batch unless nothing else is left
        else {
            break; // pool empty and no tile left (otherwise the refill branch was taken)
        }
#undef OMERF_PICK
#pragma unroll
        for (int j = 0; j < OMERF_PJ; j++) b[j] = __ballot_sync(FULL, st_lane[j] == (uint32_t)phase);
        // ---- the slots in that state, in slot order
        {
            int base = 0;
#pragma unroll
            for (int j = 0; j < OMERF_PJ; j++) {
                const int pos = base + __popc(b[j] & lt_mask);
                if ((b[j] >> lane) & 1u) P.list[chk(pos, OMERF_POOL, CHK_LIST)] = (uint8_t)(lane + 32 * j);
                base += __popc(b[j]);
            }
        }
        __syncwarp();
        const int n_act = min(n_sel, 32);
        const bool active = lane < n_act;
        const int slot = active ? chk((int)P.list[lane], OMERF_POOL, CHK_SLOT) : 0;

        if (phase == ST_IDLE) {
            // ---- refill: one 8x4 tile -> 32 new rays (S2, S3)
            unsigned t = 0;
            if (lane == 0) t = atomicAdd(tile_counter, 1u);
            const unsigned tile = tile_first + __shfl_sync(FULL, t, 0);
            if (tile + endgame_tiles >= total_tiles) endgame = true;
            if (tile >= total_tiles) {
                more = false;
            } else {
                const unsigned view = tile / tiles_per_view, tv = tile - view * tiles_per_view;
                const int ty = (int)(tv / (unsigned)tiles_x), tx = (int)(tv - (unsigned)ty * tiles_x);
                const int u = tx * 8 + (lane & 7), v = ty * 4 + (lane >> 3);
                if (u < W && v < H) {
                    const omerf_camera cam = cams[chk(view, lb.n_views, CHK_VIEW)];
                    const size_t pix = chk(((size_t)view * H + v) * W + u, lb.n_pix, CHK_PIXEL);
                    Ray r;
                    int k, k1;
                    if (setup_ray(sc, cam, u, v, r, k, k1)) {
                        P.meta[slot] = pack_meta(ST_TRAV, start_lvl, view);
                        P.d[0][slot] = r.dx;
                        P.d[1][slot] = r.dy;
                        P.d[2][slot] = r.dz;
                        P.k[slot] = k;
                        P.k1[slot] = k1;
                        P.Q[slot] = 0;
                        P.n[slot] = 0;
                        P.pix[slot] = (uint32_t)pix;
#pragma unroll
                        for (int c = 0; c < 7; c++) P.acc[c][slot] = 0.0f;
                    } else { // cannot hit the box: background (R14)
                        out_rgb[pix * 3 + 0] = sc.bg[0];
                        out_rgb[pix * 3 + 1] = sc.bg[1];
                        out_rgb[pix * 3 + 2] = sc.bg[2];
                        out_n[pix] = 0;
                    }
                }
            }
        } else if (phase == ST_TRAV) {
            // ---- traversal visit (S4).  (Two rays per lane, interleaved dependency chains, was measured slower on
            // B200 at every threshold: 0.80-0.86 ms against 0.76 ms per configs[1] frame.)
            trav_visit<SAMPLER>(sc, P, cams, lb, oc, lane, n_sel, (more && !endgame) ? OMERF_TRAV_KEEP : OMERF_DRAIN_TRAV_KEEP, out_rgb, out_n);
        } else if (phase == ST_READY) {
            // ---- samples: gather, activations, compositing (S5, S6, S7) for the rays listed in P.list[0 .. n_sel);
            // lanes whose ray left the READY state take the next listed rays, OMERF_SAMPLE_SWAP lanes at a time
            int status = ST_IDLE, k = 0, k1 = -1, lvl = 0, sslot = -1;
            uint32_t view = 0, Q = 0, n = 0;
            float acc[7];
            Ray r;
            auto load_ray = [&](int s_new) {
                sslot = s_new;
                const int s_ = s_new < 0 ? OMERF_NO_RAY : chk(s_new, OMERF_POOL, CHK_SLOT);
                view = P.meta[s_] >> 8;
                status = s_new < 0 ? ST_IDLE : ST_READY;
                k = P.k[s_];
                k1 = P.k1[s_];
                Q = P.Q[s_];
                n = P.n[s_];
                r.dx = P.d[0][s_];
                r.dy = P.d[1][s_];
                r.dz = P.d[2][s_];
                ray_origin(oc, cams, lb, view, r);
#pragma unroll
                for (int c = 0; c < 7; c++) acc[c] = P.acc[c][s_];
            };
            auto store_ray = [&]() {
                P.k[sslot] = k;
                P.Q[sslot] = Q;
                P.n[sslot] = n;
#pragma unroll
                for (int c = 0; c < 7; c++) P.acc[c][sslot] = acc[c];
                P.meta[sslot] = pack_meta(status, lvl, view);
            };
            load_ray(active ? slot : -1);
            int next = n_act; // first list entry not yet taken
#pragma unroll 1
            while (true) {
                if (status == ST_READY) {
                    float px, py, pz;
                    lattice_point(r, sc.step, k, px, py, pz);
                    if (LOG) {
                        const unsigned at = atomicAdd(tile_counter + 32, 1u);
                        if (at < log_capacity) sample_log[at] = make_uint2(P.pix[sslot], (uint32_t)k);
                    }
                    // Inside the slab the next lattice point is usually occupied too: test it here (level 0).  The test
                    // does not depend on the features, so its pyramid load is in flight together with the gather.
                    bool next_ready = false;
                    if (SAMPLER == OMERF_SAMPLER_PLANE) {
                        float qx, qy, qz;
                        lattice_point(r, sc.step, k + 1, qx, qy, qz);
                        if (k < k1) { // k + 1 is inside the box then (setup_ray): no clamp, no box test
                            const int ix = cell_index_in_box(qx, sc.sx), iy = cell_index_in_box(qy, sc.sy);
                            const float2 h = __ldg(sc.pyr + chk((uint32_t)(ix * sc.My + iy), sc.n_pyr, CHK_PYR));
                            next_ready = h.x <= qz && qz <= h.y;
                        }
                    } else {
                        // the comparator's predicate at the next lattice point: its level-0 voxel bit (R18)
                        float qx, qy, qz;
                        lattice_point(r, sc.step, k + 1, qx, qy, qz);
                        if (k < k1)
                            next_ready = occ_test(sc, 0, voxel_index_in_box(qx, sc.ns[0], sc.N[0]), voxel_index_in_box(qy, sc.ns[1], sc.N[1]),
                                                  voxel_index_in_box(qz, sc.ns[2], sc.N[2]));
                    }
                    float soft_m = 1.0f;
                    if (GENERAL && SAMPLER == OMERF_SAMPLER_PLANE && sc.soft_eps > 0.0f) {
                        // Eq. 6 (q = 2) at the nearest grid point of P_o (Eq. 7): the sample is inside [z_min, z_max],
                        // so M = min(1, ((z - z_min)/eps)^2, ((z_max - z)/eps)^2); it weights the colours only (Eq. 8)
                        const int ix = cell_index_in_box(px, sc.sx), iy = cell_index_in_box(py, sc.sy);
                        const float2 h = __ldg(sc.pyr + chk((uint32_t)(ix * sc.My + iy), sc.n_pyr, CHK_PYR));
                        const float m = __saturatef(fminf(pz - h.x, h.y - pz) * sc.inv_soft_eps);
                        soft_m = m * m;
                    }
                    uint32_t I[8];
                    gather_features<GENERAL>(sc, px, py, pz, I);
                    float t[8];
#pragma unroll
                    for (int c = 1; c < 8; c++) t[c] = fmaf(__uint2float_rn(I[c]), sc.deq_mul_half, sc.deq_add_half); // colour path
                    t[0] = __fmaf_rn(__uint2float_rn(I[0]), sc.deq_mul, sc.deq_add);                                     // decision path
                    const float tau = exp_q(t[0]); // decision path
                    const float od = __fmul_rn(tau, sc.step);
                    const uint32_t qk = (uint32_t)rintf(fminf(__fmul_rn(od, 1048576.0f), (float)sc.q_stop));
                    const float T = __expf(-(float)Q * (1.0f / 1048576.0f)); // colour path: fast math
                    const float wgt = T * (1.0f - __expf(-od)) * soft_m;
#pragma unroll
                    for (int c = 0; c < 7; c++) acc[c] = fmaf(wgt, sigmoid_of_half(t[1 + c]), acc[c]);
                    Q += qk;
                    n += 1;
                    k += 1;
                    if (Q >= sc.q_stop) {
                        status = ST_FIN; // early stop (R7)
                    } else {
                        status = next_ready ? ST_READY : ST_TRAV;
                        lvl = 0;
                    }
                }
                const unsigned going = __ballot_sync(FULL, status == ST_READY);
                if (next < n_sel) {
                    const unsigned fm = ~going;
                    if (__popc(fm) >= OMERF_SAMPLE_SWAP) {
                        if (status != ST_READY) {
                            if (sslot >= 0) store_ray();
                            const int idx = next + __popc(fm & lt_mask);
                            load_ray(idx < n_sel ? (int)P.list[idx] : -1);
                        }
                        next = min(next + __popc(fm), n_sel);
                    }
                } else if (__popc(going) < OMERF_SAMPLE_KEEP) {
                    break;
                }
            }
            if (sslot >= 0) store_ray();
        } else {
            // ---- retire: deferred MLP on tensor cores + outputs (S8, S9)
#pragma unroll 1
            for (int half = 0; half < 2; half++) {
                if (half * 16 >= n_act) break;
                // layer-1 A fragments straight from the pool (column order of omerf_mlp.cuh): lane (g, t) makes its ten
                // values of rays g and g + 8 of this half from direction component t (t = 3: the four feature sums)
                float v[2][10], o[4];
#pragma unroll
                for (int rr = 0; rr < 2; rr++) {
                    const int ray = half * 16 + (lane >> 2) + 8 * rr, tq = lane & 3;
                    const int sl = ray < n_act ? chk((int)P.list[ray], OMERF_POOL, CHK_SLOT) : slot; // unused rows: their outputs are not read
                    mlp_encode_component<true>(P.d[min(tq, 2)][sl], v[rr]);
                    v[rr][9] = P.acc[tq][sl];
                    if (tq == 3) {
                        v[rr][0] = v[rr][9];
                        v[rr][1] = P.acc[4][sl];
                        v[rr][2] = P.acc[5][sl];
                        v[rr][3] = P.acc[6][sl];
                    }
                }
                mlp_tiles(sc.mlp_tab, v[0], v[1], lane, o);
                // lane (g, t): t = 0 holds colours 0,1 and t = 1 colour 2 of rays g and g+8 of this half
                const int g = lane >> 2, t = lane & 3;
                if (t < 2) {
#pragma unroll
                    for (int rr = 0; rr < 2; rr++) {
                        const int ray = half * 16 + g + 8 * rr;
                        if (ray < n_act) {
                            const int sl = chk((int)P.list[ray], OMERF_POOL, CHK_SLOT);
                            const size_t pix = chk((size_t)P.pix[sl], lb.n_pix, CHK_PIXEL);
                            const float T_end = __expf(-(float)P.Q[sl] * (1.0f / 1048576.0f));
                            if (t == 0) {
                                out_rgb[pix * 3 + 0] = __saturatef(P.acc[0][sl] + sigmoid_fast(o[2 * rr]) + T_end * sc.bg[0]);
                                out_rgb[pix * 3 + 1] = __saturatef(P.acc[1][sl] + sigmoid_fast(o[2 * rr + 1]) + T_end * sc.bg[1]);
                                out_n[pix] = P.n[sl];
                            } else {
                                out_rgb[pix * 3 + 2] = __saturatef(P.acc[2][sl] + sigmoid_fast(o[2 * rr]) + T_end * sc.bg[2]);
                            }
                        }
                    }
                }
                __syncwarp();
            }
            if (active) P.meta[slot] = ST_IDLE;
        }
        __syncwarp();
    }
}

// ---------------------------------------------------------------------------------- gather calibration
// Replays the 10 feature loads (4 grid + 3 x 2 plane entries, 16 bytes = two adjacent texels each) of logged samples with no filtering,
// activation or compositing: one sample per thread, every lane busy, full occupancy.  The rate it reaches is the
// gather ceiling of this scene, camera and load width on this GPU; `order` selects frame order (the order the
// march kernel took the samples) or a scattered order (multiplicative permutation of the log).
__global__ void __launch_bounds__(256)
omerf_gather_probe_kernel(const __grid_constant__ DevScene sc, const omerf_camera *__restrict__ cam, int W,
                          const uint2 *__restrict__ sample_log, unsigned int n, unsigned int mult, uint32_t *__restrict__ sink)
{
    const unsigned int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const unsigned int j = (unsigned int)(((unsigned long long)i * mult) % n);
    const uint2 e = __ldg(sample_log + j);
    const int v = (int)(e.x / (unsigned)W), u = (int)(e.x - (unsigned)v * (unsigned)W);
    Ray r;
    ray_direction(*cam, u, v, r.dx, r.dy, r.dz);
    r.ox = cam->origin[0];
    r.oy = cam->origin[1];
    r.oz = cam->origin[2];
    float px, py, pz;
    lattice_point(r, sc.step, (int)e.y, px, py, pz);
    // the same 10 sixteen-byte loads as gather_features (addresses only; weights are not needed)
    int x0, y0, z0, xa, ya, za, xb, yb, zb;
    uint32_t w;
    axis_tap(px, sc.gs[0], x0, w);
    axis_tap(py, sc.gs[1], y0, w);
    axis_tap(pz, sc.gs[2], z0, w);
    uint32_t off[4];
    grid_corner_offsets<true>(sc, x0, min(x0 + 1, sc.G[0] - 1), y0, z0, min(z0 + 1, sc.G[2] - 1), off);
    uint4 t[10];
#pragma unroll
    for (int q = 0; q < 4; q++) t[q] = __ldg(sc.grid + chk(off[q], sc.n_grid, CHK_GRID));
    axis_tap(px, sc.xy_s[0], xa, w);
    axis_tap(py, sc.xy_s[1], ya, w);
    axis_tap(px, sc.xz_s[0], xb, w);
    axis_tap(pz, sc.xz_s[1], za, w);
    axis_tap(py, sc.yz_s[0], yb, w);
    axis_tap(pz, sc.yz_s[1], zb, w);
    const uint32_t Nxy = (uint32_t)sc.xy_n[1], Nxz = (uint32_t)sc.xz_rows, Nyz = (uint32_t)sc.yz_rows;
    const uint32_t zr = (uint32_t)(za - sc.xz_zoff), zs = (uint32_t)(zb - sc.yz_zoff);
    t[4] = __ldg(sc.pxy + chk((uint32_t)xa * Nxy + (uint32_t)ya, sc.n_pxy, CHK_PXY));
    t[5] = __ldg(sc.pxy + chk((uint32_t)min(xa + 1, sc.xy_n[0] - 1) * Nxy + (uint32_t)ya, sc.n_pxy, CHK_PXY));
    t[6] = __ldg(sc.pxz + chk((uint32_t)xb * Nxz + zr, sc.n_pxz, CHK_PXZ));
    t[7] = __ldg(sc.pxz + chk((uint32_t)min(xb + 1, sc.xz_n[0] - 1) * Nxz + zr, sc.n_pxz, CHK_PXZ));
    t[8] = __ldg(sc.pyz + chk((uint32_t)yb * Nyz + zs, sc.n_pyz, CHK_PYZ));
    t[9] = __ldg(sc.pyz + chk((uint32_t)min(yb + 1, sc.yz_n[0] - 1) * Nyz + zs, sc.n_pyz, CHK_PYZ));
    uint32_t x = 0;
#pragma unroll
    for (int q = 0; q < 10; q++) x ^= (t[q].x + t[q].y) ^ (t[q].z + t[q].w);
    sink[i] = x;
}

} // namespace

int omerf_launch_gather_probe(const omerf_scene *s, const omerf_camera *d_cam, int W, const uint2 *sample_log,
                              unsigned int n, unsigned int mult, uint32_t *sink, cudaStream_t st)
{
    if (n == 0) return OMERF_OK;
    omerf_gather_probe_kernel<<<(n + 255) / 256, 256, 0, st>>>(s->dev, d_cam, W, sample_log, n, mult, sink);
    OMERF_CUDA(cudaGetLastError());
    return OMERF_OK;
}

int omerf_launch_render(const omerf_scene *s, const omerf_camera *d_cams, int n_views, int W, int H, float *out_rgb,
                        uint32_t *out_n, cudaStream_t st, unsigned int *tile_counter, int *launches, uint2 *sample_log,
                        unsigned int log_capacity, unsigned int tile_first, unsigned int tile_end)
{
    if ((long long)((W + 7) / 8) * ((H + 3) / 4) * n_views > 0x7fffffffll || (long long)W * H * n_views > 0xffffffffll) {
        omerf_set_error("invalid argument: image or batch too large");
        return OMERF_ERR_INVALID;
    }
    OMERF_CUDA(cudaMemsetAsync(tile_counter, 0, (sample_log ? OMERF_COUNTER_WORDS : 1) * sizeof(unsigned int), st));
    const unsigned int all_tiles = (unsigned int)(((W + 7) / 8) * ((H + 3) / 4)) * (unsigned int)n_views;
    if (tile_end == 0 || tile_end > all_tiles) tile_end = all_tiles; // 0: the whole batch
    if (tile_first >= tile_end) {
        *launches = 0;
        return OMERF_OK;
    }
    const int grid = s->persistent_blocks;
    const bool general = s->dev.soft_eps > 0.0f || s->dev.blk_shift != 0;
#define OMERF_LAUNCH(SAMPLER, LOG, GENERAL)                                                                                 \
    omerf_march_kernel<SAMPLER, LOG, GENERAL><<<grid, 32 * OMERF_WARPS, 0, st>>>(                                          \
        s->dev, d_cams, n_views, W, H, out_rgb, out_n, tile_counter, sample_log, log_capacity, tile_first, tile_end)
#define OMERF_LAUNCH2(SAMPLER, LOG)                \
    if (general) OMERF_LAUNCH(SAMPLER, LOG, true); \
    else OMERF_LAUNCH(SAMPLER, LOG, false)
    if (s->dev.sampler == OMERF_SAMPLER_PLANE) {
        if (sample_log) { OMERF_LAUNCH2(OMERF_SAMPLER_PLANE, true); }
        else { OMERF_LAUNCH2(OMERF_SAMPLER_PLANE, false); }
    } else {
        if (sample_log) { OMERF_LAUNCH2(OMERF_SAMPLER_GRID, true); }
        else { OMERF_LAUNCH2(OMERF_SAMPLER_GRID, false); }
    }
#undef OMERF_LAUNCH2
#undef OMERF_LAUNCH
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
        OMERF_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, omerf_march_kernel<OMERF_SAMPLER_PLANE, false, true>, 32 * OMERF_WARPS, 0));
    else
        OMERF_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, omerf_march_kernel<OMERF_SAMPLER_GRID, false, true>, 32 * OMERF_WARPS, 0));
    *blocks = sms * (per_sm > 0 ? per_sm : 1);
    return OMERF_OK;
}

// ---------------------------------------------------------------------------------------------------------------------
// omerf_render_static (include/omerf.h): the render call for callers that must not allocate.
//
// Who needs it: a frame loop with a deadline (cudaMalloc synchronises the whole device and stalls the process's other
// streams whenever omerf_render's camera ring has to grow), and a plug-in whose host program owns all device memory or
// forbids driver allocations after start-up.  What it does differently: the march kernel's scratch - the device copy of
// the cameras and the work-queue head - is not a cudaMalloc'd ring slot but the fixed array below, which is part of the
// library image.  Nothing in this section calls cudaMalloc, cudaMallocHost, cudaFree or an allocating library routine.
//
// The array: one per GPU that loads the library, 2304 B, held until the process exits, shared by every scene, stream and
// thread.  It keeps whatever the last call left in it, so every call rewrites all it reads: the cameras by the staging
// kernel, the queue head by the cudaMemsetAsync in omerf_launch_render - both in stream order ahead of the march kernel.
// Calls whose kernels can overlap on the GPU (unordered streams) race on it; the header says so.
//
// Host code must not hand `omerf_static_scratch` itself to a kernel: in host code that name is only the host-side
// stand-in of the symbol.  The device address comes from cudaGetSymbolAddress, asked once per device with that device
// current (the first call on a device does it - before any stream capture, see the header) and kept in a table.
namespace {
struct StaticScratch {
    unsigned int head[OMERF_COUNTER_WORDS];    // word 0: work-queue head of the march kernel
    omerf_camera cams[OMERF_STATIC_MAX_VIEWS]; // device copy of the call's cameras
};
struct StaticCameraArgs {                      // the cameras travel as launch arguments (2 KiB): no staging buffer,
    omerf_camera cam[OMERF_STATIC_MAX_VIEWS];  // pageable host memory is fine, read before the call returns
};
} // namespace

static __device__ __align__(256) unsigned char omerf_static_scratch[sizeof(StaticScratch)];

namespace {
__global__ void __launch_bounds__(128)
omerf_static_stage_kernel(const __grid_constant__ StaticCameraArgs args, int n_views, StaticScratch *scratch)
{
    const float *src = reinterpret_cast<const float *>(args.cam);
    float *dst = reinterpret_cast<float *>(scratch->cams);
    for (int i = (int)threadIdx.x; i < n_views * (int)(sizeof(omerf_camera) / sizeof(float)); i += (int)blockDim.x) dst[i] = src[i];
}

#define OMERF_STATIC_MAX_DEVICES 64
StaticScratch *g_static_ptr[OMERF_STATIC_MAX_DEVICES]; // device address of omerf_static_scratch, per device ordinal
} // namespace

// Device address of the array on the CURRENT device `dev`; the first call per device asks the runtime for it.
// Not locked: a scene handle is used by one host thread at a time, and two threads that race here store the same value.
static int static_scratch_address(int dev, StaticScratch **out)
{
    if (dev < 0 || dev >= OMERF_STATIC_MAX_DEVICES) {
        omerf_set_error("invalid argument: omerf_render_static supports device ordinals below %d", OMERF_STATIC_MAX_DEVICES);
        return OMERF_ERR_INVALID;
    }
    StaticScratch *p = g_static_ptr[dev];
    if (!p) {
        OMERF_CUDA(cudaGetSymbolAddress((void **)&p, omerf_static_scratch));
        g_static_ptr[dev] = p;
    }
    *out = p;
    return OMERF_OK;
}

extern "C" int omerf_render_static(const omerf_scene *s, const omerf_camera *cameras, int n_views, int W, int H,
                                   float *out_rgb, uint32_t *out_nsamples, void *stream)
{
    if (!s || !cameras || !out_rgb || !out_nsamples) {
        omerf_set_error("invalid argument: null scene/cameras/output");
        return OMERF_ERR_INVALID;
    }
    if (n_views < 0 || W <= 0 || H <= 0) {
        omerf_set_error("invalid argument: n_views >= 0, W > 0, H > 0 required");
        return OMERF_ERR_INVALID;
    }
    if (n_views > OMERF_STATIC_MAX_VIEWS) {
        omerf_set_error("invalid argument: omerf_render_static takes at most %d views per call (got %d): its scratch is a "
                        "fixed array; split the batch or use omerf_render",
                        OMERF_STATIC_MAX_VIEWS, n_views);
        return OMERF_ERR_INVALID;
    }
    if (((uintptr_t)out_rgb & 3) || ((uintptr_t)out_nsamples & 3)) {
        omerf_set_error("invalid argument: misaligned output");
        return OMERF_ERR_INVALID;
    }
    s->last_launches = 0;
    if (n_views == 0) return OMERF_OK;
    int dev = -1;
    OMERF_CUDA(cudaGetDevice(&dev));
    if (dev != s->device) {
        omerf_set_error("invalid argument: scene lives on device %d but device %d is current", s->device, dev);
        return OMERF_ERR_INVALID;
    }
    StaticScratch *scratch = nullptr;
    int rc = static_scratch_address(dev, &scratch);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    StaticCameraArgs args;
    memcpy(args.cam, cameras, (size_t)n_views * sizeof(omerf_camera));
    memset(args.cam + n_views, 0, (size_t)(OMERF_STATIC_MAX_VIEWS - n_views) * sizeof(omerf_camera));
    omerf_static_stage_kernel<<<1, 128, 0, st>>>(args, n_views, scratch);
    OMERF_CUDA(cudaGetLastError());
    int launches = 0;
    // the existing launcher, given the static array instead of a ring slot; it clears the queue head on `st` first
    rc = omerf_launch_render(s, scratch->cams, n_views, W, H, out_rgb, out_nsamples, st, scratch->head, &launches);
    s->last_launches = 1 + launches;
    return rc;
}
