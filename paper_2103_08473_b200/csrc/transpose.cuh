// Bandwidth-bound tensor transposition kernels ("A(a,c,b,d) += B(a,b,c,d)").
// complex128 elements are 16 bytes: every global access is one 16-byte vector load/store per thread, a warp
// covers 512 contiguous bytes on both the read and the write side; the 32x32 tile goes through padded shared
// memory so that neither side is strided in HBM.
#pragma once
#include "common.cuh"

constexpr int TR_TILE = 32;

// General 4-index permutation whose fastest index changes.  x runs over the input-fastest group of dims; y runs over
// ALL the dims that follow x in the output order, merged into one index (they are contiguous in the output, whatever their
// order and strides in the input: e.g. ijab -> baji is the 2-d transposition x = b, y = (a,j,i)); the dims that precede x
// in the output order are batch dims r1, r2.
struct Tr4 {
    int64_t nx, ny, n1, n2;        // extents: x, merged y, batch r1, r2
    int nsub;                      // number of sub-dims of y (1-3)
    unsigned e1, e2;               // extents of the two fastest sub-dims of y (output order; the slowest is implied)
    int64_t iy0, iy1, iy2;         // input strides of the sub-dims of y, slowest first, right-aligned (x has stride 1)
    int64_t i1, i2;                // input strides of r1, r2
    int64_t ox, o1, o2;            // output strides of x, r1, r2 (y has stride 1)
    int conj;
};

// TY = rows (y) of a tile: 32, or 40 / 48 / 64 when 32 < ny <= 64 so that one tile covers y (no nearly empty second tile row).
// CTA order inside one matrix: y fastest.  CTAs resident together then write whole runs of the same output rows (measured:
// ijab -> abij 5.49 -> 6.00 TB/s, the <ab||cd> slab transposition 6.09 -> 6.31 TB/s; x-fastest order leaves half-page writes).
template <int TY, bool MULTI>
__global__ void __launch_bounds__(256) transpose4_kernel(const c128* __restrict__ in, c128* __restrict__ out, Tr4 t)
{
    __shared__ c128 tile[TY][TR_TILE + 1];
    const int64_t ty_n = (t.ny + TY - 1) / TY, tx_n = (t.nx + TR_TILE - 1) / TR_TILE;
    int64_t b = blockIdx.x;
    const int64_t by = b % ty_n; b /= ty_n;
    const int64_t bx = b % tx_n; b /= tx_n;
    const int64_t r1 = b % t.n1, r2 = b / t.n1;
    const c128* src = in + r1 * t.i1 + r2 * t.i2;
    c128* dst = out + r1 * t.o1 + r2 * t.o2;
    const int lx = threadIdx.x % TR_TILE, ly = threadIdx.x / TR_TILE;   // 32 x 8
    // input offset of the warp's rows (a warp reads TY/8 rows, each row by all 32 lanes): with one y sub-dim it is
    // y * stride; otherwise lane r decomposes the r-th row once (32-bit mixed radix) and the loads fetch it by shuffle
    int64_t rowoff = 0;
    if (MULTI && lx < TY / 8) {
        const int64_t y = by * TY + ly + 8 * lx;
        if (y < t.ny) {
            const unsigned yy = (unsigned)y, s2 = yy % t.e2, q = yy / t.e2, s1 = q % t.e1, s0 = q / t.e1;
            rowoff = s0 * t.iy0 + s1 * t.iy1 + s2 * t.iy2;
        }
    }
#pragma unroll
    for (int k = 0; k < TY; k += 8) {
        const int64_t x = bx * TR_TILE + lx, y = by * TY + ly + k;
        const int64_t off = MULTI ? __shfl_sync(0xffffffffu, rowoff, k / 8) : y * t.iy2;
        if (x < t.nx && y < t.ny) {
            c128 val = src[off + x];
            if (t.conj) val.y = -val.y;
            tile[ly + k][lx] = val;
        }
    }
    __syncthreads();
    if (TY > TR_TILE) {
        // one tile covers y (ny <= TY) and, with ox == ny, the CTA's output is ONE contiguous run of (its x count) * ny
        // elements: written linearly (512-byte warps) instead of ny-element rows split into a 32-lane and a ragged pass
        const unsigned ny = (unsigned)t.ny;
        const int64_t xleft = t.nx - bx * TR_TILE;
        const unsigned count = (unsigned)(xleft < TR_TILE ? xleft : TR_TILE) * ny;
        c128* run = dst + bx * TR_TILE * t.ox;
        if (t.ox == t.ny) {
            for (unsigned e = threadIdx.x; e < count; e += 256) {
                const unsigned xx = e / ny, yy = e - xx * ny;
                run[e] = tile[yy][xx];
            }
            return;
        }
    }
#pragma unroll
    for (int yy = 0; yy < TY; yy += TR_TILE) {
#pragma unroll
        for (int k = 0; k < TR_TILE; k += 8) {
            const int64_t y = by * TY + yy + lx, x = bx * TR_TILE + ly + k;
            if (x < t.nx && y < t.ny) dst[x * t.ox + y] = tile[yy + lx][ly + k];
        }
    }
}
template <int TY>
static inline void launch_tr4_ty(cudaStream_t st, const c128* in, c128* out, const Tr4& t, unsigned blocks)
{
    if (t.nsub > 1) transpose4_kernel<TY, true><<<blocks, 256, 0, st>>>(in, out, t);
    else transpose4_kernel<TY, false><<<blocks, 256, 0, st>>>(in, out, t);
}
static inline int launch_tr4(cudaStream_t st, const c128* in, c128* out, const Tr4& t)
{
    // 32 < ny <= 64 (an occupied index, typically): one tile of 40, 48 or 64 rows covers y
    const int ty = (t.ny <= TR_TILE || t.ny > 64) ? TR_TILE : t.ny <= 40 ? 40 : t.ny <= 48 ? 48 : 64;
    const int64_t blocks = ((t.nx + TR_TILE - 1) / TR_TILE) * ((t.ny + ty - 1) / ty) * t.n1 * t.n2;
    if (blocks > 0x7fffffffLL) return CCSD_EINVAL;
    if (blocks == 0) return CCSD_OK;
    switch (ty) {
    case 40: launch_tr4_ty<40>(st, in, out, t, (unsigned)blocks); break;
    case 48: launch_tr4_ty<48>(st, in, out, t, (unsigned)blocks); break;
    case 64: launch_tr4_ty<64>(st, in, out, t, (unsigned)blocks); break;
    default: launch_tr4_ty<TR_TILE>(st, in, out, t, (unsigned)blocks); break;
    }
    return CCSD_OK;
}

// Fastest index preserved: the tensor is a set of contiguous rows of nx elements that are re-ordered.  The kernel
// walks the OUTPUT linearly (perfectly coalesced 16-byte stores, 8 independent 16-byte loads in flight per thread) and
// decomposes the output row index into the (up to three) slow output dims to find the input row.
struct Cp4 {
    int64_t nx, total;             // row length, total elements
    unsigned n1, n2;               // extents of the two fastest slow OUTPUT dims (n0 is implied)
    int64_t i0, i1, i2;            // input strides of the slow output dims
    int conj;
};
constexpr int CP_UNROLL = 8;
__global__ void __launch_bounds__(256) copy4_kernel(const c128* __restrict__ in, c128* __restrict__ out, Cp4 t)
{
    const int64_t base = (int64_t)blockIdx.x * (256 * CP_UNROLL);
    // 64-bit division once per block; everything below is 32-bit relative to the block's first row
    const int64_t row0 = base / t.nx;
    const unsigned x0 = (unsigned)(base - row0 * t.nx), nx = (unsigned)t.nx;
    const int64_t q0 = row0 / t.n2, a0_0 = q0 / t.n1;
    const unsigned a2_0 = (unsigned)(row0 - q0 * t.n2), a1_0 = (unsigned)(q0 - a0_0 * t.n1);
    c128 val[CP_UNROLL];
#pragma unroll
    for (int k = 0; k < CP_UNROLL; k++) {
        const unsigned off = x0 + threadIdx.x + 256u * k;
        if (base + threadIdx.x + 256 * k < t.total) {
            const unsigned drow = off / nx, x = off - drow * nx;         // rows past the block's first one (< 2048 + 1)
            const unsigned s2 = a2_0 + drow, c2 = s2 / t.n2, a2 = s2 - c2 * t.n2;   // mixed-radix increment with carries
            const unsigned s1 = a1_0 + c2, c1 = s1 / t.n1, a1 = s1 - c1 * t.n1;
            val[k] = in[(a0_0 + c1) * t.i0 + a1 * t.i1 + a2 * t.i2 + x];
        }
    }
#pragma unroll
    for (int k = 0; k < CP_UNROLL; k++) {
        const int64_t e = base + threadIdx.x + 256 * k;
        if (e < t.total) {
            c128 w = val[k];
            if (t.conj) w.y = -w.y;
            out[e] = w;
        }
    }
}

// out[c*ld_out + r] = in[r*ld_in + c]
static inline int launch_transpose2d_ld(cudaStream_t st, const c128* in, int64_t ld_in, c128* out, int64_t ld_out,
                                        int64_t rows, int64_t cols, int conj)
{
    if (rows <= 0 || cols <= 0) return CCSD_OK;
    Tr4 t;
    t.nx = cols; t.ny = rows; t.n1 = 1; t.n2 = 1;
    t.nsub = 1; t.e1 = 1; t.e2 = (unsigned)1; t.iy0 = 0; t.iy1 = 0; t.iy2 = ld_in;
    t.i1 = 0; t.i2 = 0;
    t.ox = ld_out; t.o1 = 0; t.o2 = 0;
    t.conj = conj;
    CCSD_TRY(launch_tr4(st, in, out, t));
    count_launches(1);
    CCSD_CUDA_TRY(cudaGetLastError());
    return CCSD_OK;
}
static inline int launch_transpose2d(cudaStream_t st, const c128* in, c128* out, int64_t rows, int64_t cols, int conj)
{
    return launch_transpose2d_ld(st, in, cols, out, rows, rows, cols, conj);
}

// out dimension q is input dimension perm[q].  Extent-1 dims are dropped and input dims that stay adjacent (in the same
// order) in the output are merged first, so that e.g. ijab -> abij runs as ONE 2-d transposition (ij) x (ab) with full
// tiles instead of o x v ragged ones.
static inline int launch_transpose4d(cudaStream_t st, const c128* in, c128* out, const int64_t d[4], const int perm[4], int conj)
{
    int seen[4] = {0, 0, 0, 0};
    for (int q = 0; q < 4; q++) {
        if (perm[q] < 0 || perm[q] > 3 || seen[perm[q]]) return CCSD_EINVAL;
        seen[perm[q]] = 1;
        if (d[q] < 0) return CCSD_EINVAL;
    }
    const int64_t total = d[0] * d[1] * d[2] * d[3];
    if (total == 0) return CCSD_OK;
    // rank of every non-trivial input dim in the output order
    int orank[4] = {-1, -1, -1, -1}, nout = 0;
    for (int q = 0; q < 4; q++)
        if (d[perm[q]] > 1) orank[perm[q]] = nout++;
    // groups of merged dims, in input order
    int ng = 0, grank[4];
    int64_t gext[4];
    for (int q = 0, prev = -1; q < 4; q++) {
        if (d[q] <= 1) continue;
        if (prev >= 0 && orank[q] == orank[prev] + 1) {
            gext[ng - 1] *= d[q];
        } else {
            gext[ng] = d[q]; grank[ng] = orank[q]; ng++;
        }
        prev = q;
    }
    if (ng == 0) { ng = 1; gext[0] = 1; grank[0] = 0; }
    // input strides (groups are in input order) and the groups in output order
    int64_t gis[4], gos[4];
    gis[ng - 1] = 1;
    for (int k = ng - 2; k >= 0; k--) gis[k] = gis[k + 1] * gext[k + 1];
    int order[4];   // order[r] = group that is r-th in the output
    for (int r = 0; r < ng; r++) {
        int best = -1;
        for (int k = 0; k < ng; k++) {
            bool used = false;
            for (int rr = 0; rr < r; rr++) used |= (order[rr] == k);
            if (!used && (best < 0 || grank[k] < grank[best])) best = k;
        }
        order[r] = best;
    }
    gos[order[ng - 1]] = 1;
    for (int r = ng - 2; r >= 0; r--) gos[order[r]] = gos[order[r + 1]] * gext[order[r + 1]];

    if (order[ng - 1] == ng - 1) {
        // fastest group preserved: re-ordered contiguous rows
        Cp4 t;
        t.nx = gext[ng - 1]; t.total = total; t.conj = conj;
        int64_t ext[3] = {1, 1, 1}, ist[3] = {0, 0, 0};   // slow output dims, right-aligned
        for (int r = ng - 2, s = 2; r >= 0; r--, s--) { ext[s] = gext[order[r]]; ist[s] = gis[order[r]]; }
        if (ext[1] > 0xffffffffLL || ext[2] > 0xffffffffLL || t.nx > 0x7fffffffLL) return CCSD_EINVAL;
        t.n1 = (unsigned)ext[1]; t.n2 = (unsigned)ext[2];
        t.i0 = ist[0]; t.i1 = ist[1]; t.i2 = ist[2];
        const int64_t blocks = (total + 256 * CP_UNROLL - 1) / (256 * CP_UNROLL);
        if (blocks > 0x7fffffffLL) return CCSD_EINVAL;
        copy4_kernel<<<(unsigned)blocks, 256, 0, st>>>(in, out, t);
    } else {
        // x: the input-fastest group, at position px of the output order; y: every group after px (contiguous in the
        // output), merged; the groups before px are batch dims
        const int gx = ng - 1;
        int px = 0;
        while (order[px] != gx) px++;
        Tr4 t;
        t.nx = gext[gx]; t.ox = gos[gx];
        t.ny = 1;
        int64_t ye[3] = {1, 1, 1}, yi[3] = {0, 0, 0};     // sub-dims of y, slowest first, right-aligned
        t.nsub = 0;
        for (int r = ng - 1, sidx = 2; r > px; r--, sidx--) { ye[sidx] = gext[order[r]]; yi[sidx] = gis[order[r]]; t.ny *= gext[order[r]]; t.nsub++; }
        if (t.nsub > 1 && t.ny > 0xffffffffLL) return CCSD_EINVAL;   // 32-bit mixed radix (> 64 GB per x: not reachable)
        t.e1 = (unsigned)ye[1]; t.e2 = (unsigned)ye[2];
        t.iy0 = yi[0]; t.iy1 = yi[1]; t.iy2 = yi[2];
        t.n1 = 1; t.n2 = 1; t.i1 = t.i2 = t.o1 = t.o2 = 0;
        for (int r = px - 1, nr = 0; r >= 0; r--, nr++) {   // r1 (the faster CTA index) = the batch dim next to x in the output
            const int k = order[r];
            if (nr == 0) { t.n1 = gext[k]; t.i1 = gis[k]; t.o1 = gos[k]; }
            else { t.n2 = gext[k]; t.i2 = gis[k]; t.o2 = gos[k]; }
        }
        t.conj = conj;
        CCSD_TRY(launch_tr4(st, in, out, t));
    }
    count_launches(1);
    CCSD_CUDA_TRY(cudaGetLastError());
    return CCSD_OK;
}
