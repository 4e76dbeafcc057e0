/*
 * omerf_oracle.c — CPU ORACLE of the Oblique-MERF render hot path.
 *
 * THIS FILE IS TEST INFRASTRUCTURE.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may build, load or call it.
 * It shares no code, header, table or constant generator with the CUDA path
 * (paper_2404_09531_b200/csrc, include/omerf.h) and neither includes the other.
 *
 * What it computes (readings R1..R20; citations are
 * /root/reference/PAPER.md line numbers):
 *   - per pixel a pinhole ray r = o + t d                         PAPER.md:63  (sec. 3)
 *   - a fixed lattice of samples t_k = (k + 1/2) step             reading R4/R5
 *   - sample kept iff inside the box and inside the occupancy
 *     interval [z_min, z_max] of the NEAREST grid point of P_o     PAPER.md:104, :116-118 (Eq. 7), :137
 *   - features t(p) = V(p) + P_xy(p) + P_xz(p) + P_yz(p)           PAPER.md:69-72 (Eq. 2)
 *   - tau = exp(t0), c^d = sigmoid(t1..3), f = sigmoid(t4..7)      PAPER.md:74-77 (Eq. 3)
 *   - C = sum_i w_i c_i, w_i = T_i alpha_i, alpha = 1 - e^{-tau d} PAPER.md:65-67 (Eq. 1), :122 (Eq. 8, binary M)
 *   - C = sum w c^d + G([sum w c^d, sum w f], d)                   PAPER.md:79-81 (Eq. 4)
 *   - optional soft occupancy M of Eq. 6 (q = 2) weighting w_i       PAPER.md:114-122 (Eq. 6-8), SURVEY 8(f).2
 * The occupancy-plane *marching* of PAPER.md:188 is an exact acceleration (it
 * reaches the same samples), so it does NOT appear here: the oracle is the plain
 * definition — every lattice sample tested with the per-sample predicate.
 *
 * Precision.  Everything that decides an INTEGER (which samples exist, when the
 * ray terminates: out_nsamples) is computed in fp32 with one correctly rounded
 * IEEE operation per step (fmaf / * / + / / / sqrtf / rintf / floorf), or in
 * exact integer arithmetic, so that the CUDA kernels can take the same decisions
 * in the same precision.  Build with -ffp-contract=off and without fast-math.
 * Everything else (activations, compositing, MLP: out_rgb) is fp64.
 *
 * Two loop forms that must agree bit for bit: BRUTE (all k in [0,K)) and
 * CLIPPED (k-range from a double-precision box intersection padded by 2
 * indices on both sides; the predicate is unchanged).
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): closed-form slab transmittance,
 * empty scene == background, sum of weights == 1 - T_end, brute == clipped,
 * interpolation vs scipy.ndimage.map_coordinates, exp_q vs libm exp, MLP vs
 * numpy float64 matmul, x<->y transpose symmetry, step refinement, bitfield
 * popcount vs analytic slab volume, n_grid >= n_plane.
 * Conventions the paper does not fix (R4 lattice phase, R10 texel addressing,
 * R13 MLP activations/encoding, R19 camera) are "parity unpinned by the paper":
 * pinned only by DESIGN.md.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    float box[3];                       /* world box [0,X]x[0,Y]x[0,Z], z up */
    int32_t hf_n[2];                    /* Mx, My grid points of the occupancy plane */
    const float *h_lo, *h_up;           /* [Mx][My] z_min, z_max */
    int32_t grid_n[3];
    const uint8_t *grid;                /* [Gx][Gy][Gz][8] */
    int32_t xy_n[2], xz_n[2], yz_n[2];
    const uint8_t *plane_xy, *plane_xz, *plane_yz; /* [A][B][8] */
    float deq_scale, deq_bias;          /* value = u8*scale + bias (R12) */
    int32_t mlp_in, mlp_hidden;         /* 34, 16 */
    const float *W0, *b0, *W1, *b1, *W2, *b2; /* row-major [out][in] */
    float step, t_stop, bg[3];
    int32_t sampler;                    /* 0 occupancy plane, 1 binary occupancy grid (config 4) */
    int32_t occ_n[3];
    const uint32_t *occ_bits;           /* sampler 1: bit index ((jx*Ny+jy)*Nz+jz), LSB-first words */
    float soft_eps;                     /* > 0: soft occupancy function of Eq. 6 with buffer eps; 0: binary mask */
} orc_scene;

typedef struct {
    float origin[3], right[3], up[3], fwd[3];
    float fx, fy, cx, cy;
} orc_camera;

/* ------------------------------------------------------------------ exp_q (R8) */
/* Reproducible fp32 exponential: accuracy is irrelevant, every step is one
 * correctly rounded operation.  Cody-Waite reduction + degree-6 Taylor/Horner. */
float orc_exp_q(float x)
{
    float y = x * 0x1.715476p+0f;             /* x * log2(e) */
    float n = rintf(y);
    float f = fmaf(n, -0x1.62e4p-1f, x);      /* x - n*ln2_hi */
    f = fmaf(n, -0x1.7f7d1cp-20f, f);         /*   - n*ln2_lo */
    float p = (float)(1.0 / 720.0);
    p = fmaf(p, f, (float)(1.0 / 120.0));
    p = fmaf(p, f, (float)(1.0 / 24.0));
    p = fmaf(p, f, (float)(1.0 / 6.0));
    p = fmaf(p, f, 0.5f);
    p = fmaf(p, f, 1.0f);
    p = fmaf(p, f, 1.0f);
    int32_t e = (int32_t)n + 127;             /* |x| <= 87 keeps 1 <= e <= 254 */
    if (e < 1) e = 1;
    if (e > 254) e = 254;
    uint32_t bits = (uint32_t)e << 23;
    float scale;
    memcpy(&scale, &bits, 4);
    return p * scale;                          /* exact scaling by 2^n */
}

/* Q_STOP = ceil(-ln(t_stop) * 2^20), in double (R7/R8). 7243307 for t_stop = 1e-3. */
uint32_t orc_q_stop(float t_stop)
{
    return (uint32_t)ceil(-log((double)t_stop) * 1048576.0);
}

/* ------------------------------------------------------------------ ray (R19, sec. 8(b) pixel convention) */
void orc_ray(const orc_camera *c, int u, int v, float d[3])
{
    float a = ((float)u + 0.5f - c->cx) / c->fx;
    float b = -(((float)v + 0.5f - c->cy) / c->fy);
    float g[3];
    for (int i = 0; i < 3; i++) g[i] = fmaf(a, c->right[i], fmaf(b, c->up[i], c->fwd[i]));
    float len2 = fmaf(g[0], g[0], fmaf(g[1], g[1], g[2] * g[2]));
    float inv = 1.0f / sqrtf(len2);
    for (int i = 0; i < 3; i++) d[i] = g[i] * inv;
}

/* lattice sample k (R4): t_k = (k + 1/2) step, p = o + t_k d, one fma per component */
static inline void lattice_point(const float o[3], const float d[3], float step, int64_t k, float p[3])
{
    float t = ((float)k + 0.5f) * step;
    for (int i = 0; i < 3; i++) p[i] = fmaf(t, d[i], o[i]);
}

static inline int in_box(const orc_scene *s, const float p[3])
{
    return p[0] >= 0.0f && p[0] < s->box[0] && p[1] >= 0.0f && p[1] < s->box[1] &&
           p[2] >= 0.0f && p[2] < s->box[2];
}

static inline int clampi(int v, int lo, int hi) { return v < lo ? lo : (v > hi ? hi : v); }

/* ------------------------------------------------------------------ predicates */
/* Eq. 7: nearest grid point of P_o; closed interval (R1, R2, R3). */
int orc_occupied_plane(const orc_scene *s, const float p[3])
{
    int Mx = s->hf_n[0], My = s->hf_n[1];
    float sx = (float)(Mx - 1) / s->box[0];
    float sy = (float)(My - 1) / s->box[1];
    int ix = clampi((int)floorf(fmaf(p[0], sx, 0.5f)), 0, Mx - 1);
    int iy = clampi((int)floorf(fmaf(p[1], sy, 0.5f)), 0, My - 1);
    float lo = s->h_lo[(size_t)ix * My + iy];
    float hi = s->h_up[(size_t)ix * My + iy];
    return lo <= p[2] && p[2] <= hi;
}

/* Soft occupancy function M of Eq. 6, exponent q = 2, evaluated at the nearest grid
 * point of P_o (Eq. 7).  Written as the paper's four cases; where the two buffer zones overlap (interval thinner than
 * 2 eps - the paper is silent, R23) the smaller of the two ramps is taken, which keeps M continuous. */
double orc_soft_mask(const orc_scene *s, const float p[3])
{
    int Mx = s->hf_n[0], My = s->hf_n[1];
    float sx = (float)(Mx - 1) / s->box[0];
    float sy = (float)(My - 1) / s->box[1];
    int ix = clampi((int)floorf(fmaf(p[0], sx, 0.5f)), 0, Mx - 1);
    int iy = clampi((int)floorf(fmaf(p[1], sy, 0.5f)), 0, My - 1);
    double zmin = (double)s->h_lo[(size_t)ix * My + iy], zmax = (double)s->h_up[(size_t)ix * My + iy];
    double z = (double)p[2], eps = (double)s->soft_eps;
    if (z < zmin || z > zmax) return 0.0;                         /* second case of Eq. 6 */
    if (!(eps > 0.0)) return 1.0;                                 /* binary mask (R3) */
    double m = 1.0;                                               /* first case */
    if (z <= zmin + eps) { double a = (z - zmin) / eps; m = a * a; }          /* third case, q = 2 */
    if (z >= zmax - eps) { double b = (zmax - z) / eps; if (b * b < m) m = b * b; } /* fourth case */
    return m;
}

/* config-4 comparator: binary occupancy grid (the structure PAPER.md:188 replaces). */
int orc_occupied_grid(const orc_scene *s, const float p[3])
{
    int Nx = s->occ_n[0], Ny = s->occ_n[1], Nz = s->occ_n[2];
    int jx = (int)floorf(p[0] * ((float)Nx / s->box[0]));
    int jy = (int)floorf(p[1] * ((float)Ny / s->box[1]));
    int jz = (int)floorf(p[2] * ((float)Nz / s->box[2]));
    if (jx > Nx - 1) jx = Nx - 1;
    if (jy > Ny - 1) jy = Ny - 1;
    if (jz > Nz - 1) jz = Nz - 1;
    if (jx < 0) jx = 0;
    if (jy < 0) jy = 0;
    if (jz < 0) jz = 0;
    uint64_t idx = ((uint64_t)jx * Ny + jy) * Nz + jz;
    return (s->occ_bits[idx >> 5] >> (idx & 31)) & 1u;
}

/* Bitfield derivation (R18): voxel set iff its closed z-range intersects the closed
 * interval [h_lo,h_up] of ANY occupancy cell whose xy square overlaps the voxel's xy
 * square with positive area.  Cell i spans [(i-1/2), (i+1/2)] X/(Mx-1); voxel j spans
 * [j, j+1] X/Nx; overlap tests in exact integers, z tests in double. */
/* first/last cell i (inclusive) overlapping voxel j with positive length along one axis:
 * 2 j (M-1) < (2i+1) N  and  (2i-1) N < 2 (j+1) (M-1)   (exact integers) */
static void cell_range(int j, int N, int M, int *i0, int *i1)
{
    int lo = -1, hi = -2;
    for (int i = 0; i < M; i++) {
        int64_t a = 2 * (int64_t)j * (M - 1), b = (2 * (int64_t)i + 1) * N;
        int64_t c = (2 * (int64_t)i - 1) * N, e = 2 * ((int64_t)j + 1) * (M - 1);
        if (a < b && c < e) {
            if (lo < 0) lo = i;
            hi = i;
        } else if (lo >= 0) break;
    }
    *i0 = lo;
    *i1 = hi;
}

void orc_build_bitfield(const orc_scene *s, uint32_t *bits)
{
    int Nx = s->occ_n[0], Ny = s->occ_n[1], Nz = s->occ_n[2];
    int Mx = s->hf_n[0], My = s->hf_n[1];
    size_t nwords = ((size_t)Nx * Ny * Nz + 31) / 32;
    memset(bits, 0, nwords * 4);
    double Z = (double)s->box[2];
    int *xr = (int *)malloc(sizeof(int) * 2 * (size_t)Nx);
    int *yr = (int *)malloc(sizeof(int) * 2 * (size_t)Ny);
    /* cell ranges are monotone in j, but M is small: a plain search per j is fine */
    for (int j = 0; j < Nx; j++) cell_range(j, Nx, Mx, &xr[2 * j], &xr[2 * j + 1]);
    for (int j = 0; j < Ny; j++) cell_range(j, Ny, My, &yr[2 * j], &yr[2 * j + 1]);
#pragma omp parallel for schedule(static)
    for (int jx = 0; jx < Nx; jx++) {
        for (int jy = 0; jy < Ny; jy++) {
            for (int jz = 0; jz < Nz; jz++) {
                double zl = ((double)jz * Z) / (double)Nz;
                double zh = ((double)(jz + 1) * Z) / (double)Nz;
                int set = 0;
                for (int ix = xr[2 * jx]; ix <= xr[2 * jx + 1] && !set; ix++)
                    for (int iy = yr[2 * jy]; iy <= yr[2 * jy + 1] && !set; iy++) {
                        double lo = (double)s->h_lo[(size_t)ix * My + iy];
                        double hi = (double)s->h_up[(size_t)ix * My + iy];
                        if (lo <= hi && zl <= hi && zh >= lo) set = 1;
                    }
                if (set) {
                    uint64_t idx = ((uint64_t)jx * Ny + jy) * Nz + jz;
#pragma omp atomic
                    bits[idx >> 5] |= 1u << (idx & 31);
                }
            }
        }
    }
    free(xr);
    free(yr);
}

/* ------------------------------------------------------------------ features (Eq. 2, R9, R10) */
/* One axis: texel coordinate q = p*N/X - 1/2 (texel centres at (i+1/2) X/N), lower
 * texel i0 = floor(q), 8-bit weight w = floor(frac*256 + 1/2) in [0,256], clamp-to-edge. */
static inline void axis_tap(float p, int N, float X, int *i0, int *i1, uint32_t *w)
{
    float q = fmaf(p, (float)N / X, -0.5f);
    float fl = floorf(q);
    *w = (uint32_t)(int)floorf((q - fl) * 256.0f + 0.5f);
    int i = (int)fl;
    *i0 = clampi(i, 0, N - 1);
    *i1 = clampi(i + 1, 0, N - 1);
}

/* bilinear tap sum over axes (a,b) of tex[Na][Nb][8] with 8-bit weights: exact integers <= 255*2^16 */
static inline void bilinear8(const uint8_t *tex, int Nb, int a0, int a1, uint32_t wa, int b0, int b1,
                             uint32_t wb, uint32_t B[8])
{
    const uint8_t *t00 = tex + ((size_t)a0 * Nb + b0) * 8;
    const uint8_t *t10 = tex + ((size_t)a1 * Nb + b0) * 8;
    const uint8_t *t01 = tex + ((size_t)a0 * Nb + b1) * 8;
    const uint8_t *t11 = tex + ((size_t)a1 * Nb + b1) * 8;
    for (int c = 0; c < 8; c++)
        B[c] = (256u - wa) * (256u - wb) * t00[c] + wa * (256u - wb) * t10[c] +
               (256u - wa) * wb * t01[c] + wa * wb * t11[c];
}

/* public wrapper for the interpolation pin: plane lookup at (pa, pb) */
void orc_plane_lookup(const uint8_t *tex, int Na, int Nb, float Xa, float Xb, float pa, float pb,
                      uint32_t B[8])
{
    int a0, a1, b0, b1;
    uint32_t wa, wb;
    axis_tap(pa, Na, Xa, &a0, &a1, &wa);
    axis_tap(pb, Nb, Xb, &b0, &b1, &wb);
    bilinear8(tex, Nb, a0, a1, wa, b0, b1, wb, B);
}

/* grid lookup: bilinear in (x,y) on the two z-slices, then I_V = ((256-wz) B0 + wz B1 + 128) >> 8 */
void orc_grid_lookup(const uint8_t *grid, const int32_t G[3], const float box[3], const float p[3],
                     uint32_t I[8])
{
    int x0, x1, y0, y1, z0, z1;
    uint32_t wx, wy, wz;
    axis_tap(p[0], G[0], box[0], &x0, &x1, &wx);
    axis_tap(p[1], G[1], box[1], &y0, &y1, &wy);
    axis_tap(p[2], G[2], box[2], &z0, &z1, &wz);
    for (int c = 0; c < 8; c++) {
        uint32_t Bz[2];
        for (int s = 0; s < 2; s++) {
            int z = s ? z1 : z0;
            uint32_t t00 = grid[(((size_t)x0 * G[1] + y0) * G[2] + z) * 8 + c];
            uint32_t t10 = grid[(((size_t)x1 * G[1] + y0) * G[2] + z) * 8 + c];
            uint32_t t01 = grid[(((size_t)x0 * G[1] + y1) * G[2] + z) * 8 + c];
            uint32_t t11 = grid[(((size_t)x1 * G[1] + y1) * G[2] + z) * 8 + c];
            Bz[s] = (256u - wx) * (256u - wy) * t00 + wx * (256u - wy) * t10 +
                    (256u - wx) * wy * t01 + wx * wy * t11;
        }
        I[c] = ((256u - wz) * Bz[0] + wz * Bz[1] + 128u) >> 8;
    }
}

/* t(p) = V(p) + P_xy(p) + P_xz(p) + P_yz(p)  (Eq. 2), as integers I (units of u8 * 2^16)
 * and dequantised pre-activations t_c = fma(I, scale/65536, 4*bias) in fp32. */
void orc_features(const orc_scene *s, const float p[3], int32_t I[8], float t[8])
{
    uint32_t V[8], Pxy[8], Pxz[8], Pyz[8];
    orc_grid_lookup(s->grid, s->grid_n, s->box, p, V);
    orc_plane_lookup(s->plane_xy, s->xy_n[0], s->xy_n[1], s->box[0], s->box[1], p[0], p[1], Pxy);
    orc_plane_lookup(s->plane_xz, s->xz_n[0], s->xz_n[1], s->box[0], s->box[2], p[0], p[2], Pxz);
    orc_plane_lookup(s->plane_yz, s->yz_n[0], s->yz_n[1], s->box[1], s->box[2], p[1], p[2], Pyz);
    float mul = s->deq_scale / 65536.0f;
    float add = 4.0f * s->deq_bias;
    for (int c = 0; c < 8; c++) {
        I[c] = (int32_t)(V[c] + Pxy[c] + Pxz[c] + Pyz[c]);
        t[c] = fmaf((float)I[c], mul, add);
    }
}

/* ------------------------------------------------------------------ deferred MLP (Eq. 4, R13) */
static inline double sigmoid_d(double x) { return 1.0 / (1.0 + exp(-x)); }

/* enc(d) = [d, then for j=0..3, for c=x,y,z: sin(2^j d_c), cos(2^j d_c)]  (27 values) */
void orc_encode_dir(const float d[3], double enc[27])
{
    int n = 0;
    for (int c = 0; c < 3; c++) enc[n++] = (double)d[c];
    for (int j = 0; j < 4; j++)
        for (int c = 0; c < 3; c++) {
            double a = (double)(1 << j) * (double)d[c];
            enc[n++] = sin(a);
            enc[n++] = cos(a);
        }
}

/* G: in(34) -> relu(16) -> relu(16) -> sigmoid(3), fp64 accumulation of the fp32 weights */
void orc_mlp(const orc_scene *s, const double *in, double out[3])
{
    int ni = s->mlp_in, nh = s->mlp_hidden;
    double h1[64], h2[64];
    for (int o = 0; o < nh; o++) {
        double a = (double)s->b0[o];
        for (int i = 0; i < ni; i++) a += (double)s->W0[o * ni + i] * in[i];
        h1[o] = a > 0.0 ? a : 0.0;
    }
    for (int o = 0; o < nh; o++) {
        double a = (double)s->b1[o];
        for (int i = 0; i < nh; i++) a += (double)s->W1[o * nh + i] * h1[i];
        h2[o] = a > 0.0 ? a : 0.0;
    }
    for (int o = 0; o < 3; o++) {
        double a = (double)s->b2[o];
        for (int i = 0; i < nh; i++) a += (double)s->W2[o * nh + i] * h2[i];
        out[o] = sigmoid_d(a);
    }
}

/* ------------------------------------------------------------------ render (Eq. 1, 4, 8; R4..R8, R14, R15) */
typedef struct {
    double rgb[3];
    uint32_t n;
    double T_end, sum_w;
    uint32_t Q;
} orc_pixel;

/* K: no lattice index >= K can be inside the box (R4): K = ceil((|o - c| + diag/2)/step) + 1, in double */
int64_t orc_lattice_K(const orc_scene *s, const orc_camera *cam)
{
    double c[3] = {0.5 * s->box[0], 0.5 * s->box[1], 0.5 * s->box[2]};
    double dist = 0.0, diag = 0.0;
    for (int i = 0; i < 3; i++) {
        double e = (double)cam->origin[i] - c[i];
        dist += e * e;
        diag += (double)s->box[i] * (double)s->box[i];
    }
    return (int64_t)ceil((sqrt(dist) + 0.5 * sqrt(diag)) / (double)s->step) + 1;
}

/* CLIPPED form only: k-range from a double-precision slab test, padded by 2 on both sides */
static void clipped_range(const orc_scene *s, const float o[3], const float d[3], int64_t K,
                          int64_t *k0, int64_t *k1)
{
    double t0 = 0.0, t1 = INFINITY;
    for (int i = 0; i < 3; i++) {
        double oi = o[i], di = d[i], hi = s->box[i];
        if (di == 0.0) {
            if (oi < 0.0 || oi > hi) { *k0 = 0; *k1 = -1; return; }
        } else {
            double a = (0.0 - oi) / di, b = (hi - oi) / di;
            if (a > b) { double t = a; a = b; b = t; }
            if (a > t0) t0 = a;
            if (b < t1) t1 = b;
        }
    }
    if (t0 > t1) { *k0 = 0; *k1 = -1; return; }
    double st = (double)s->step;
    int64_t a = (int64_t)floor(t0 / st - 0.5) - 2;
    int64_t b = (int64_t)ceil(t1 / st - 0.5) + 2;
    if (a < 0) a = 0;
    if (b > K - 1) b = K - 1;
    *k0 = a;
    *k1 = b;
}

/* ------------------------------------------------------------------ compulsory bytes */
/* Distinct 32-byte sectors of the four feature arrays ([..][8] uint8, row-major as in the scene) touched by the samples
 * of a render: the bytes a cache of unbounded size would still have to fetch once.  Bit maps (one bit per sector) are
 * installed by orc_set_sector_maps and filled by the render loops; maps[0] = grid, 1 = xy, 2 = xz, 3 = yz. */
static uint8_t *g_sector_map[4] = {0, 0, 0, 0};

void orc_set_sector_maps(uint8_t *grid, uint8_t *xy, uint8_t *xz, uint8_t *yz)
{
    g_sector_map[0] = grid;
    g_sector_map[1] = xy;
    g_sector_map[2] = xz;
    g_sector_map[3] = yz;
}

static inline void mark_texel(uint8_t *map, size_t texel)
{
    size_t sector = texel >> 2;                              /* 8-byte texels, 32-byte sectors */
    uint8_t bit = (uint8_t)(1u << (sector & 7));
    if (!(map[sector >> 3] & bit)) {
#pragma omp atomic
        map[sector >> 3] |= bit;
    }
}

static void mark_sample_sectors(const orc_scene *s, const float p[3])
{
    int a0, a1, b0, b1, c0, c1;
    uint32_t w;
    axis_tap(p[0], s->grid_n[0], s->box[0], &a0, &a1, &w);
    axis_tap(p[1], s->grid_n[1], s->box[1], &b0, &b1, &w);
    axis_tap(p[2], s->grid_n[2], s->box[2], &c0, &c1, &w);
    const int xs[2] = {a0, a1}, ys[2] = {b0, b1}, zs[2] = {c0, c1};
    for (int i = 0; i < 2; i++)
        for (int j = 0; j < 2; j++)
            for (int k = 0; k < 2; k++)
                mark_texel(g_sector_map[0], ((size_t)xs[i] * s->grid_n[1] + ys[j]) * s->grid_n[2] + zs[k]);
    const int32_t *pn[3] = {s->xy_n, s->xz_n, s->yz_n};
    const int ax[3][2] = {{0, 1}, {0, 2}, {1, 2}};
    for (int q = 0; q < 3; q++) {
        axis_tap(p[ax[q][0]], pn[q][0], s->box[ax[q][0]], &a0, &a1, &w);
        axis_tap(p[ax[q][1]], pn[q][1], s->box[ax[q][1]], &b0, &b1, &w);
        const int as[2] = {a0, a1}, bs[2] = {b0, b1};
        for (int i = 0; i < 2; i++)
            for (int j = 0; j < 2; j++) mark_texel(g_sector_map[1 + q], (size_t)as[i] * pn[q][1] + bs[j]);
    }
}

static void render_pixel(const orc_scene *s, const orc_camera *cam, int u, int v, int64_t K, int mode,
                         uint32_t q_stop, orc_pixel *out)
{
    float d[3], o[3] = {cam->origin[0], cam->origin[1], cam->origin[2]};
    orc_ray(cam, u, v, d);
    int64_t k0 = 0, k1 = K - 1;
    if (mode == 1) clipped_range(s, o, d, K, &k0, &k1);

    uint32_t Q = 0, n = 0;
    double D[3] = {0, 0, 0}, Fs[4] = {0, 0, 0, 0}, sum_w = 0.0;
    for (int64_t k = k0; k <= k1; k++) {
        float p[3];
        lattice_point(o, d, s->step, k, p);
        if (!in_box(s, p)) continue;
        int occ = s->sampler == 0 ? orc_occupied_plane(s, p) : orc_occupied_grid(s, p);
        if (!occ) continue;                                   /* Eq. 8 with binary M (R3) */
        if (Q >= q_stop) break;                               /* early stop, tested before the sample (R7) */
        int32_t I[8];
        float t[8];
        orc_features(s, p, I, t);                             /* Eq. 2 */
        if (g_sector_map[0]) mark_sample_sectors(s, p);
        float tau = orc_exp_q(t[0]);                          /* Eq. 3, decision path */
        float od = tau * s->step;                             /* tau_i * delta_i, delta = step (R5) */
        uint32_t qk = (uint32_t)rintf(fminf(od * 1048576.0f, (float)q_stop));
        double T = exp(-(double)Q * (1.0 / 1048576.0));       /* T_i = prod_{j<i}(1 - alpha_j) (R6) */
        double alpha = 1.0 - exp(-(double)od);
        double w = T * alpha;                                 /* omega_i = T_i alpha_i (Eq. 1) */
        /* Eq. 8: the contribution of sample i is M_i omega_i c_i; M = 1 inside the interval for the binary mask */
        double Mw = (s->soft_eps > 0.0f && s->sampler == 0) ? orc_soft_mask(s, p) * w : w;
        for (int c = 0; c < 3; c++) D[c] += Mw * sigmoid_d((double)t[1 + c]);
        for (int c = 0; c < 4; c++) Fs[c] += Mw * sigmoid_d((double)t[4 + c]);
        sum_w += w;
        Q += qk;
        n += 1;
    }
    double T_end = exp(-(double)Q * (1.0 / 1048576.0));
    out->n = n;
    out->T_end = T_end;
    out->sum_w = sum_w;
    out->Q = Q;
    if (n == 0) {                                             /* R14: empty ray == background exactly */
        for (int c = 0; c < 3; c++) out->rgb[c] = (double)s->bg[c];
        return;
    }
    double in[64], S[3];
    for (int c = 0; c < 3; c++) in[c] = D[c];
    for (int c = 0; c < 4; c++) in[3 + c] = Fs[c];
    orc_encode_dir(d, in + 7);
    orc_mlp(s, in, S);                                        /* Eq. 4 */
    for (int c = 0; c < 3; c++) {
        double x = D[c] + S[c] + T_end * (double)s->bg[c];
        out->rgb[c] = x < 0.0 ? 0.0 : (x > 1.0 ? 1.0 : x);
    }
}

/* Render rows [v_begin, v_end) of every view.  mode 0 = BRUTE, 1 = CLIPPED.
 * out_rgb  double [n_views][H][W][3], out_n uint32 [n_views][H][W] (rows outside the range untouched),
 * out_aux  double [n_views][H][W][3] = (T_end, sum of weights, Q) or NULL,
 * view_total uint64 [n_views] or NULL, hist uint64 [64] samples/ray histogram (last bin = 63+) or NULL.
 * Returns the number of OpenMP threads used. */
int orc_render(const orc_scene *s, const orc_camera *cams, int n_views, int W, int H, int v_begin,
               int v_end, int mode, double *out_rgb, uint32_t *out_n, double *out_aux,
               uint64_t *view_total, uint64_t *hist)
{
    uint32_t q_stop = orc_q_stop(s->t_stop);
    int nthreads = 1;
    if (hist) memset(hist, 0, 64 * sizeof(uint64_t));
    for (int view = 0; view < n_views; view++) {
        const orc_camera *cam = cams + view;
        int64_t K = orc_lattice_K(s, cam);
        uint64_t total = 0;
        uint64_t h[64];
        memset(h, 0, sizeof h);
#pragma omp parallel
        {
            uint64_t lt = 0, lh[64];
            memset(lh, 0, sizeof lh);
#ifdef _OPENMP
#pragma omp single
            nthreads = omp_get_num_threads();
#endif
#pragma omp for schedule(dynamic, 1)
            for (int v = v_begin; v < v_end; v++) {
                for (int u = 0; u < W; u++) {
                    orc_pixel px;
                    render_pixel(s, cam, u, v, K, mode, q_stop, &px);
                    size_t idx = ((size_t)view * H + v) * W + u;
                    for (int c = 0; c < 3; c++) out_rgb[idx * 3 + c] = px.rgb[c];
                    out_n[idx] = px.n;
                    if (out_aux) {
                        out_aux[idx * 3 + 0] = px.T_end;
                        out_aux[idx * 3 + 1] = px.sum_w;
                        out_aux[idx * 3 + 2] = (double)px.Q;
                    }
                    lt += px.n;
                    lh[px.n < 63 ? px.n : 63]++;
                }
            }
#pragma omp critical
            {
                total += lt;
                for (int i = 0; i < 64; i++) h[i] += lh[i];
            }
        }
        if (view_total) view_total[view] = total;
        if (hist) for (int i = 0; i < 64; i++) hist[i] += h[i];
    }
    return nthreads;
}

/* Render a list of pixels (view, u, v triples) — parity on sampled outputs at full size.
 * out_rgb double [n_pix][3], out_n uint32 [n_pix], out_aux double [n_pix][3] or NULL. */
int orc_render_pixels(const orc_scene *s, const orc_camera *cams, int n_views, int W, int H, int mode,
                      int64_t n_pix, const int32_t *vuv, double *out_rgb, uint32_t *out_n, double *out_aux)
{
    uint32_t q_stop = orc_q_stop(s->t_stop);
    int64_t *Ks = (int64_t *)malloc(sizeof(int64_t) * (size_t)n_views);
    for (int i = 0; i < n_views; i++) Ks[i] = orc_lattice_K(s, cams + i);
    int bad = 0;
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t i = 0; i < n_pix; i++) {
        int view = vuv[3 * i], u = vuv[3 * i + 1], v = vuv[3 * i + 2];
        if (view < 0 || view >= n_views || u < 0 || u >= W || v < 0 || v >= H) {
#pragma omp atomic write
            bad = 1;
            continue;
        }
        orc_pixel px;
        render_pixel(s, cams + view, u, v, Ks[view], mode, q_stop, &px);
        for (int c = 0; c < 3; c++) out_rgb[i * 3 + c] = px.rgb[c];
        out_n[i] = px.n;
        if (out_aux) {
            out_aux[i * 3 + 0] = px.T_end;
            out_aux[i * 3 + 1] = px.sum_w;
            out_aux[i * 3 + 2] = (double)px.Q;
        }
    }
    free(Ks);
    return bad ? -1 : 0;
}

/* The lattice samples of one pixel, for pins that need positions: writes up to `cap` kept sample
 * indices k and their (x,y,z); returns the number kept (ignores early stop; predicate only). */
int64_t orc_pixel_samples(const orc_scene *s, const orc_camera *cam, int u, int v, int64_t cap,
                          int64_t *ks, float *pos)
{
    float d[3], o[3] = {cam->origin[0], cam->origin[1], cam->origin[2]};
    orc_ray(cam, u, v, d);
    int64_t K = orc_lattice_K(s, cam), n = 0;
    for (int64_t k = 0; k < K; k++) {
        float p[3];
        lattice_point(o, d, s->step, k, p);
        if (!in_box(s, p)) continue;
        int occ = s->sampler == 0 ? orc_occupied_plane(s, p) : orc_occupied_grid(s, p);
        if (!occ) continue;
        if (n < cap) {
            ks[n] = k;
            pos[3 * n] = p[0]; pos[3 * n + 1] = p[1]; pos[3 * n + 2] = p[2];
        }
        n++;
    }
    return n;
}

/* ------------------------------------------------------------------ sparse-block grid */
/* the low-resolution voxel grid is stored as sparse blocks; PAPER.md:258 (sec. 5.3): the baked
 * assets are produced from the occupancy plane, which says where features can ever be fetched.  The oracle states
 * the bake as a plain rule (R24):
 *   a voxel (i,j,k) of V is NEEDED iff it can be one of the 8 trilinear corners (R10 addressing) of a point whose
 *   nearest grid point of P_o is (ix,iy) and whose z lies in [z_min, z_max](ix,iy) - with the cell footprint widened
 *   by 1/64 of a cell on every side and the z interval by 1/64 of a voxel (both far above the fp32 rounding of the
 *   renderer's coordinates, so every corner the renderer touches is needed);
 *   a B^3 block is ALLOCATED iff it holds a needed voxel; blocks are numbered in C order of (bx,by,bz);
 *   the atlas stores the allocated blocks' voxels ([id][B][B][B][8], zeros beyond the grid edge).
 * Rendering through (table, atlas) fetches exactly the dense grid's texels, so the image is the dense oracle's. */
static int64_t floordiv64(int64_t a, int64_t b) /* b > 0 */
{
    int64_t q = a / b;
    return (a % b != 0 && a < 0) ? q - 1 : q;
}

/* corner index range [lo,hi] along one horizontal axis for occupancy cell i (exact integers):
 * q = x G/X - 1/2 at x = (i -+ 33/64) X/(M-1)  ->  q = (2 (64 i -+ 33) G - 64 (M-1)) / (128 (M-1)) */
static void cell_corner_range(int i, int M, int G, int *lo, int *hi)
{
    int64_t den = 128 * (int64_t)(M - 1);
    int64_t a = floordiv64(2 * (64 * (int64_t)i - 33) * G - 64 * (int64_t)(M - 1), den);
    int64_t b = floordiv64(2 * (64 * (int64_t)i + 33) * G - 64 * (int64_t)(M - 1), den) + 1;
    *lo = (int)(a < 0 ? 0 : a);
    *hi = (int)(b > G - 1 ? G - 1 : b);
}

/* needed z-corner range of one column, in double with one rounding per operation; returns 0 if none */
static int column_corner_range(float lo, float hi, float Z, int G, int *k_lo, int *k_hi)
{
    if (!(lo <= hi)) return 0;                                /* empty column (R17) */
    double zl = lo < 0.0f ? 0.0 : (double)lo, zh = hi > Z ? (double)Z : (double)hi;
    if (zl > zh) return 0;                                    /* interval outside the box */
    double qa = zl * (double)G / (double)Z - 0.515625;        /* - 1/2 - 1/64 */
    double qb = zh * (double)G / (double)Z - 0.484375;        /* - 1/2 + 1/64 */
    int64_t a = (int64_t)floor(qa), b = (int64_t)floor(qb) + 1;
    *k_lo = (int)(a < 0 ? 0 : a);
    *k_hi = (int)(b > G - 1 ? G - 1 : b);
    return 1;
}

/* needed-voxel mask, uint8 [Gx][Gy][Gz] (tiny scenes / pins only) */
void orc_sparse_need_mask(const orc_scene *s, uint8_t *need)
{
    const int Mx = s->hf_n[0], My = s->hf_n[1], Gx = s->grid_n[0], Gy = s->grid_n[1], Gz = s->grid_n[2];
    memset(need, 0, (size_t)Gx * Gy * Gz);
    for (int ix = 0; ix < Mx; ix++)
        for (int iy = 0; iy < My; iy++) {
            int i0, i1, j0, j1, k0, k1;
            if (!column_corner_range(s->h_lo[(size_t)ix * My + iy], s->h_up[(size_t)ix * My + iy], s->box[2], Gz, &k0, &k1))
                continue;
            cell_corner_range(ix, Mx, Gx, &i0, &i1);
            cell_corner_range(iy, My, Gy, &j0, &j1);
            for (int i = i0; i <= i1; i++)
                for (int j = j0; j <= j1; j++)
                    for (int k = k0; k <= k1; k++) need[((size_t)i * Gy + j) * Gz + k] = 1;
        }
}

/* block marks uint8 [nbx][nby][nbz], nb = ceil(G/B); returns the number of allocated blocks */
int64_t orc_sparse_mark_blocks(const orc_scene *s, int B, uint8_t *mark)
{
    const int Mx = s->hf_n[0], My = s->hf_n[1], Gx = s->grid_n[0], Gy = s->grid_n[1], Gz = s->grid_n[2];
    const int nbx = (Gx + B - 1) / B, nby = (Gy + B - 1) / B, nbz = (Gz + B - 1) / B;
    memset(mark, 0, (size_t)nbx * nby * nbz);
    for (int ix = 0; ix < Mx; ix++)
        for (int iy = 0; iy < My; iy++) {
            int i0, i1, j0, j1, k0, k1;
            if (!column_corner_range(s->h_lo[(size_t)ix * My + iy], s->h_up[(size_t)ix * My + iy], s->box[2], Gz, &k0, &k1))
                continue;
            cell_corner_range(ix, Mx, Gx, &i0, &i1);
            cell_corner_range(iy, My, Gy, &j0, &j1);
            for (int bx = i0 / B; bx <= i1 / B; bx++)
                for (int by = j0 / B; by <= j1 / B; by++)
                    for (int bz = k0 / B; bz <= k1 / B; bz++) mark[((size_t)bx * nby + by) * nbz + bz] = 1;
        }
    int64_t n = 0;
    for (size_t i = 0; i < (size_t)nbx * nby * nbz; i++) n += mark[i];
    return n;
}

/* table int32 [nbx*nby*nbz]: block id (rank among the allocated blocks in C order) or -1;
 * atlas uint8 [n_alloc][B][B][B][8] (may be NULL to build the table only) */
void orc_sparse_build(const orc_scene *s, int B, const uint8_t *mark, int32_t *table, uint8_t *atlas)
{
    const int Gx = s->grid_n[0], Gy = s->grid_n[1], Gz = s->grid_n[2];
    const int nbx = (Gx + B - 1) / B, nby = (Gy + B - 1) / B, nbz = (Gz + B - 1) / B;
    int32_t id = 0;
    for (int bx = 0; bx < nbx; bx++)
        for (int by = 0; by < nby; by++)
            for (int bz = 0; bz < nbz; bz++) {
                size_t b = ((size_t)bx * nby + by) * nbz + bz;
                if (!mark[b]) {
                    table[b] = -1;
                    continue;
                }
                table[b] = id;
                if (atlas) {
                    uint8_t *dst = atlas + (size_t)id * B * B * B * 8;
                    for (int x = 0; x < B; x++)
                        for (int y = 0; y < B; y++)
                            for (int z = 0; z < B; z++) {
                                int gx = bx * B + x, gy = by * B + y, gz = bz * B + z;
                                uint8_t *t = dst + (((size_t)x * B + y) * B + z) * 8;
                                if (gx < Gx && gy < Gy && gz < Gz)
                                    memcpy(t, s->grid + (((size_t)gx * Gy + gy) * Gz + gz) * 8, 8);
                                else
                                    memset(t, 0, 8);
                            }
                }
                id++;
            }
}

/* the 8 trilinear corners of p: c = {x0, x1, y0, y1, z0, z1} (R10) */
void orc_grid_corners(const int32_t G[3], const float box[3], const float p[3], int32_t c[6])
{
    uint32_t w;
    int a, b;
    for (int ax = 0; ax < 3; ax++) {
        axis_tap(p[ax], G[ax], box[ax], &a, &b, &w);
        c[2 * ax] = a;
        c[2 * ax + 1] = b;
    }
}

/* orc_grid_lookup through (table, atlas); returns -1 if a corner lies in an unallocated block */
int orc_sparse_grid_lookup(const int32_t *table, const uint8_t *atlas, int B, const int32_t G[3], const float box[3],
                           const float p[3], uint32_t I[8])
{
    int x0, x1, y0, y1, z0, z1;
    uint32_t wx, wy, wz;
    axis_tap(p[0], G[0], box[0], &x0, &x1, &wx);
    axis_tap(p[1], G[1], box[1], &y0, &y1, &wy);
    axis_tap(p[2], G[2], box[2], &z0, &z1, &wz);
    const int nby = (G[1] + B - 1) / B, nbz = (G[2] + B - 1) / B;
    const int xs[2] = {x0, x1}, ys[2] = {y0, y1}, zs[2] = {z0, z1};
    const uint8_t *t[2][2][2];
    for (int a = 0; a < 2; a++)
        for (int b = 0; b < 2; b++)
            for (int c = 0; c < 2; c++) {
                int32_t id = table[((size_t)(xs[a] / B) * nby + ys[b] / B) * nbz + zs[c] / B];
                if (id < 0) return -1;
                t[a][b][c] = atlas + ((((size_t)id * B + xs[a] % B) * B + ys[b] % B) * B + zs[c] % B) * 8;
            }
    for (int c = 0; c < 8; c++) {
        uint32_t Bz[2];
        for (int sl = 0; sl < 2; sl++)
            Bz[sl] = (256u - wx) * (256u - wy) * t[0][0][sl][c] + wx * (256u - wy) * t[1][0][sl][c] +
                     (256u - wx) * wy * t[0][1][sl][c] + wx * wy * t[1][1][sl][c];
        I[c] = ((256u - wz) * Bz[0] + wz * Bz[1] + 128u) >> 8;
    }
    return 0;
}

/* ------------------------------------------------------------------ low-z triplane bake (second half) */
/* PAPER.md:186 (sec. 4.4): "For the 2D triplane, we employ a texture map with high resolution in the xy direction and
 * low resolution in the z direction, according to the upper and lower bounds of the occupancy plane.  This approach
 * saves a significant amount of video memory during real-time rendering."  The paper gives no rule; reading R27
 * (DESIGN.md): the xz and yz planes keep ONE contiguous band of z-texel rows [b_lo, b_hi] - the rows that a bilinear
 * lookup (R10 addressing: q = z Nz/Z - 1/2, taps floor(q) and floor(q)+1, clamped to the plane) can touch for
 *     z in [z_lo, z_hi],  z_lo = min z_min,  z_hi = max z_max  over the NON-EMPTY columns of P_o (R17), clipped to [0,Z],
 * widened by 1/64 texel on both sides (far above the fp32 rounding of the renderer's q; same padding as R24).
 * Every sample of the occupancy-plane sampler has z in [z_lo, z_hi] (Eq. 7), so no row outside the band is ever fetched
 * and the image is the uncropped oracle's.  A scene with no non-empty column keeps row 0 only (never fetched).
 * Double arithmetic, one rounding per operation.  Returns the number of rows kept. */
int orc_lowz_band(const orc_scene *s, int Nz, int *b_lo, int *b_hi)
{
    const int Mx = s->hf_n[0], My = s->hf_n[1];
    const double Z = (double)s->box[2];
    double zl = 0.0, zh = 0.0;
    int any = 0;
    for (size_t i = 0; i < (size_t)Mx * My; i++) {
        float lo = s->h_lo[i], hi = s->h_up[i];
        if (!(lo <= hi)) continue;                            /* empty column (R17) */
        if (!any || (double)lo < zl) zl = (double)lo;
        if (!any || (double)hi > zh) zh = (double)hi;
        any = 1;
    }
    if (zl < 0.0) zl = 0.0;
    if (zh > Z) zh = Z;
    if (!any || zl > zh) {
        *b_lo = 0;
        *b_hi = 0;
        return 1;
    }
    double qa = zl * (double)Nz / Z - 0.515625;               /* - 1/2 - 1/64 */
    double qb = zh * (double)Nz / Z - 0.484375;               /* - 1/2 + 1/64 */
    int64_t a = (int64_t)floor(qa), b = (int64_t)floor(qb) + 1;
    *b_lo = (int)(a < 0 ? 0 : a);
    *b_hi = (int)(b > Nz - 1 ? Nz - 1 : b);
    return *b_hi - *b_lo + 1;
}

/* the baked plane: out[Na][b_hi-b_lo+1][8] = tex[Na][b_lo..b_hi][8] */
void orc_lowz_crop(const uint8_t *tex, int Na, int Nb, int b_lo, int b_hi, uint8_t *out)
{
    const int Bk = b_hi - b_lo + 1;
    for (int a = 0; a < Na; a++)
        for (int b = 0; b < Bk; b++) memcpy(out + ((size_t)a * Bk + b) * 8, tex + ((size_t)a * Nb + b_lo + b) * 8, 8);
}

/* orc_plane_lookup through the baked band (taps addressed as in the full plane of Nb rows, then shifted by b_lo);
 * returns -1 if a z-tap of (pa, pz) lies outside the band */
int orc_plane_lookup_band(const uint8_t *band, int Na, int Nb, int b_lo, int b_hi, float Xa, float Z, float pa,
                          float pz, uint32_t B[8])
{
    int a0, a1, b0, b1;
    uint32_t wa, wb;
    axis_tap(pa, Na, Xa, &a0, &a1, &wa);
    axis_tap(pz, Nb, Z, &b0, &b1, &wb);
    if (b0 < b_lo || b1 > b_hi) return -1;
    bilinear8(band, b_hi - b_lo + 1, a0, a1, wa, b0 - b_lo, b1 - b_lo, wb, B);
    return 0;
}

/* ------------------------------------------------------------------ view-direction smoothness term */
/* PAPER.md:145-155, Eq. 9-10: for a viewing direction d, perturbed directions s = d + delta (delta ~ N(0, Sigma) is an
 * INPUT here: the random draws are the caller's) and
 *     l(d) = sum_s S(d, s) || G(F, s) - G(F, d) ||_2^2,     S = cosine similarity,
 * the forward pass of the regulariser as a batched workload of the deferred MLP G (Eq. 4).
 * Readings (R25): s is fed to the direction encoding as it is (not re-normalised; the cosine carries the
 * norms), F is the 7-vector [sum w c^d, sum w f] of Eq. 4, G's output is its three sigmoid colours.
 *   F double-free inputs: F float [n][7], d float [n][3], delta float [n][S][3]; s_c = d_c + delta_c in fp32 (one add).
 *   out_loss double [n]; out_G double [n][S+1][3] or NULL (row 0 = G(F,d)). */
void orc_mlp_smoothness(const orc_scene *s, int64_t n, int S, const float *F, const float *d, const float *delta,
                        double *out_loss, double *out_G)
{
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; i++) {
        double in[64], G0[3], Gs[3];
        for (int c = 0; c < 7; c++) in[c] = (double)F[i * 7 + c];
        const float *di = d + i * 3;
        orc_encode_dir(di, in + 7);
        orc_mlp(s, in, G0);
        if (out_G) for (int c = 0; c < 3; c++) out_G[(i * (S + 1)) * 3 + c] = G0[c];
        double loss = 0.0;
        for (int j = 0; j < S; j++) {
            float sv[3];
            for (int c = 0; c < 3; c++) sv[c] = di[c] + delta[(i * S + j) * 3 + c];
            orc_encode_dir(sv, in + 7);
            orc_mlp(s, in, Gs);
            double dot = 0.0, nd = 0.0, ns = 0.0, diff2 = 0.0;
            for (int c = 0; c < 3; c++) {
                dot += (double)di[c] * (double)sv[c];
                nd += (double)di[c] * (double)di[c];
                ns += (double)sv[c] * (double)sv[c];
                diff2 += (Gs[c] - G0[c]) * (Gs[c] - G0[c]);
            }
            double cosv = (nd > 0.0 && ns > 0.0) ? dot / sqrt(nd * ns) : 0.0;   /* S(d, s) */
            loss += cosv * diff2;
            if (out_G) for (int c = 0; c < 3; c++) out_G[(i * (S + 1) + j + 1) * 3 + c] = Gs[c];
        }
        out_loss[i] = loss;
    }
}
