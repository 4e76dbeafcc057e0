// omerf_sparse.cu — sparse-block storage of the low-resolution voxel grid V, baked from the occupancy plane
// (SURVEY.md 8(f).1; PAPER.md:186 "sparse blocks", :258 baking from the occupancy plane; R24).
//
// A voxel of V is needed iff it can be a trilinear corner of a point inside the slab: for every non-empty column
// (ix,iy) of P_o the corner ranges of the cell footprint (widened by 1/64 cell, exact integer arithmetic) and of
// [z_min, z_max] (widened by 1/64 voxel, double with one rounding per operation) are marked.  A B^3 block is
// allocated iff it holds a needed voxel; allocated blocks are numbered in C order of (bx,by,bz) by a scan and their
// voxels copied into the atlas [id][B][B][B] (16-byte entries: the texel and its +y neighbour).  The render kernels then address V through the block
// table (one indirection per corner) and fetch exactly the texels of the dense grid.
#include "omerf_device.cuh"

namespace {

__device__ __forceinline__ long long floordiv64(long long a, long long b) // b > 0
{
    long long q = a / b;
    return (a % b != 0 && a < 0) ? q - 1 : q;
}

// corner index range along one horizontal axis for occupancy cell i:
// q = x G/X - 1/2 at x = (i -+ 33/64) X/(M-1)  ->  q = (2 (64 i -+ 33) G - 64 (M-1)) / (128 (M-1))
__device__ __forceinline__ void cell_corner_range(int i, int M, int G, int &lo, int &hi)
{
    const long long den = 128ll * (M - 1);
    const long long a = floordiv64(2 * (64ll * i - 33) * G - 64ll * (M - 1), den);
    const long long b = floordiv64(2 * (64ll * i + 33) * G - 64ll * (M - 1), den) + 1;
    lo = (int)(a < 0 ? 0 : a);
    hi = (int)(b > G - 1 ? G - 1 : b);
}

__global__ void sparse_mark_kernel(const __grid_constant__ DevScene sc, int shift, int nby, int nbz, uint32_t *__restrict__ mark)
{
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= sc.Mx * sc.My) return;
    const int ix = c / sc.My, iy = c - ix * sc.My;
    const float2 h = sc.pyr[c]; // level 0 of the pyramid is P_o itself
    if (!(h.x <= h.y)) return;  // empty column (R17)
    const double Z = (double)sc.box[2];
    const double zl = h.x < 0.0f ? 0.0 : (double)h.x, zh = h.y > sc.box[2] ? Z : (double)h.y;
    if (zl > zh) return;
    const int Gz = sc.G[2];
    const double qa = __dsub_rn(__ddiv_rn(__dmul_rn(zl, (double)Gz), Z), 0.515625);
    const double qb = __dsub_rn(__ddiv_rn(__dmul_rn(zh, (double)Gz), Z), 0.484375);
    const long long ka = (long long)floor(qa), kb = (long long)floor(qb) + 1;
    const int k0 = (int)(ka < 0 ? 0 : ka), k1 = (int)(kb > Gz - 1 ? Gz - 1 : kb);
    int i0, i1, j0, j1;
    cell_corner_range(ix, sc.Mx, sc.G[0], i0, i1);
    cell_corner_range(iy, sc.My, sc.G[1], j0, j1);
    for (int bx = i0 >> shift; bx <= (i1 >> shift); bx++)
        for (int by = j0 >> shift; by <= (j1 >> shift); by++)
            for (int bz = k0 >> shift; bz <= (k1 >> shift); bz++) mark[((size_t)bx * nby + by) * nbz + bz] = 1u;
}

// exclusive scan of the marks in C order -> block ids; one CTA, every thread owns a contiguous chunk
__global__ void __launch_bounds__(1024) sparse_scan_kernel(const uint32_t *__restrict__ mark, int32_t *__restrict__ table,
                                                           unsigned int n, unsigned int *__restrict__ n_alloc)
{
    __shared__ unsigned int sums[1024];
    const unsigned int chunk = (n + 1023u) / 1024u, t = threadIdx.x;
    const unsigned int a = min(t * chunk, n), b = min(a + chunk, n);
    unsigned int s = 0;
    for (unsigned int i = a; i < b; i++) s += mark[i];
    sums[t] = s;
    __syncthreads();
    for (unsigned int d = 1; d < 1024; d <<= 1) { // Hillis-Steele inclusive scan of the chunk sums
        const unsigned int v = t >= d ? sums[t - d] : 0u;
        __syncthreads();
        sums[t] += v;
        __syncthreads();
    }
    unsigned int id = sums[t] - s;
    for (unsigned int i = a; i < b; i++) table[i] = mark[i] ? (int32_t)id++ : -1;
    if (t == 1023) *n_alloc = sums[1023];
}

// one CTA per block of the block grid; allocated blocks copy their B^3 ENTRIES (zeros past the grid edge).  An entry is
// the texel pair (y, min(y + 1, Gy - 1)) of the dense array (S0 layout, omerf_build.cu): the second texel of a block's last
// y layer comes from the neighbouring block, so the trilinear gather needs one table lookup per (x, z) corner pair.
__global__ void sparse_copy_kernel(const uint2 *__restrict__ dense, int Gx, int Gy, int Gz, int shift, int nby, int nbz,
                                   const int32_t *__restrict__ table, uint4 *__restrict__ atlas)
{
    const int32_t id = table[blockIdx.x];
    if (id < 0) return;
    const int bz = blockIdx.x % nbz, by = (blockIdx.x / nbz) % nby, bx = blockIdx.x / (nbz * nby);
    const int B = 1 << shift, m = B - 1, vox = B * B * B;
    for (int v = threadIdx.x; v < vox; v += blockDim.x) {
        const int z = v & m, y = (v >> shift) & m, x = v >> (2 * shift);
        const int gx = (bx << shift) + x, gy = (by << shift) + y, gz = (bz << shift) + z;
        uint4 t = make_uint4(0u, 0u, 0u, 0u);
        if (gx < Gx && gy < Gy && gz < Gz) {
            const size_t row = (size_t)gx * Gy;
            t = pair_entry(dense[(row + gy) * Gz + gz], dense[(row + min(gy + 1, Gy - 1)) * Gz + gz]);
        }
        atlas[(size_t)id * vox + v] = t;
    }
}

} // namespace

// Builds (block table, atlas) from the raw dense texels *d_dense ([Gx][Gy][Gz] of 8 bytes; freed here and replaced by the
// atlas); fills the sparse fields of s->dev.
int omerf_bake_sparse_grid(omerf_scene *s, void **d_dense, int block, cudaStream_t st)
{
    DevScene &v = s->dev;
    int shift = 0;
    while ((1 << shift) < block) shift++;
    const int nbx = (v.G[0] + block - 1) >> shift, nby = (v.G[1] + block - 1) >> shift, nbz = (v.G[2] + block - 1) >> shift;
    const unsigned long long nb = (unsigned long long)nbx * nby * nbz;
    if (nb > 0x7fffffffull) {
        omerf_set_error("invalid argument: too many grid blocks");
        return OMERF_ERR_INVALID;
    }
    uint32_t *mark = nullptr;
    unsigned int *d_n = nullptr, n_alloc = 0;
    int rc = OMERF_OK;
    do {
        cudaError_t e;
#define SP_CUDA(call)                                          \
    if ((e = (call)) != cudaSuccess) {                         \
        rc = omerf_cuda_fail(e, #call);                        \
        break;                                                 \
    }
        SP_CUDA(cudaMalloc((void **)&mark, nb * sizeof(uint32_t)));
        SP_CUDA(cudaMalloc((void **)&d_n, sizeof(unsigned int)));
        SP_CUDA(cudaMalloc(&s->d_blk_table, nb * sizeof(int32_t)));
        SP_CUDA(cudaMemsetAsync(mark, 0, nb * sizeof(uint32_t), st));
        const int cells = v.Mx * v.My;
        sparse_mark_kernel<<<(cells + 255) / 256, 256, 0, st>>>(v, shift, nby, nbz, mark);
        sparse_scan_kernel<<<1, 1024, 0, st>>>(mark, (int32_t *)s->d_blk_table, (unsigned int)nb, d_n);
        SP_CUDA(cudaGetLastError());
        SP_CUDA(cudaMemcpyAsync(&n_alloc, d_n, sizeof n_alloc, cudaMemcpyDeviceToHost, st));
        SP_CUDA(cudaStreamSynchronize(st));
        const unsigned long long texels = (unsigned long long)n_alloc << (3 * shift);
        if (texels > 0xffffffffull) {
            omerf_set_error("invalid argument: sparse atlas has more than 2^32 - 1 texels");
            rc = OMERF_ERR_INVALID;
            break;
        }
        void *atlas = nullptr;
        SP_CUDA(cudaMalloc(&atlas, (texels ? texels : 1) * sizeof(uint4)));
        if (n_alloc)
            sparse_copy_kernel<<<(unsigned int)nb, 256, 0, st>>>((const uint2 *)*d_dense, v.G[0], v.G[1], v.G[2], shift, nby, nbz,
                                                                 (const int32_t *)s->d_blk_table, (uint4 *)atlas);
        e = cudaGetLastError();
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        if (e != cudaSuccess) {
            cudaFree(atlas);
            rc = omerf_cuda_fail(e, "sparse_copy_kernel");
            break;
        }
#undef SP_CUDA
        cudaFree(*d_dense);
        *d_dense = atlas;
        v.grid = (const uint4 *)atlas;
        v.blk_shift = shift;
        v.nby = nby;
        v.nbz = nbz;
        v.blk_table = (const int32_t *)s->d_blk_table;
        v.n_blk = (uint32_t)nb;
        v.n_grid = (uint32_t)texels;
        s->blocks_total = nb;
        s->blocks_allocated = n_alloc;
        s->grid_bytes = texels * sizeof(uint4) + nb * sizeof(int32_t);
    } while (0);
    cudaFree(mark);
    cudaFree(d_n);
    return rc;
}
