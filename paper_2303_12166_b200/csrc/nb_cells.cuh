// nb_cells.cuh -- row a3: the contact pairs of Eqs. 5/6 through a
// CELL LIST, rebuilt from scratch at every force evaluation (the result is a function of the state alone,
// so restarts stay bitwise).  Included after nb_kernels.cuh (uses its DevState, ContactArgs, contact_term).
//
// Each star s has its own grid of cubic cells of edge h_s = max(2 R_s, R_0 + R_1): at least the reach of
// any pair that involves an element of s, so a query touches <= 3 cells per axis, and no larger than needed
// for the star with the smaller elements (with the packing of the configs, ~1.2 elements per cell of 2 R:
// the 27 cells of a query hold ~33 candidates for ~5 contacts).  Cell coordinates are counted from the
// star's mean position (robust against a few far outliers) and WRAPPED onto a table of mx x my x mz buckets,
// powers of two >= 4 with at most cap_s (2-4 n_s) buckets: the cells of a query are then distinct buckets,
// x-adjacent cells are adjacent buckets (one range of the sorted array per row of a query), and elements far
// outside the table merely alias onto it (more candidates, same pairs: which pairs ARE in contact is decided
// by contact_term() in fp64).  Containment needs no slack beyond the rounding of R_i + R_j: rounding,
// subtraction of the origin, scaling, floor and clamping are all monotone, so x_i - D <= x_j <= x_i + D puts
// j's cell inside i's range of cells on every axis.
//
//   nb_cell_bbox_kernel     per-star bounding boxes and coordinate sums (block partials); zeroes the counters
//   nb_cell_count_kernel    grid geometry (every block, from the partials); bucket of every element and
//                           its arrival number there (integer atomics: the COUNTS are deterministic)
//   nb_cell_scan_kernel x2  exclusive prefix sum of the counts -> first sorted position of every bucket
//   nb_cell_scatter_kernel  element index -> its bucket's range, in arrival order
//   nb_cell_rank_kernel     ... re-ranked by element index inside the bucket (a fixed order, whatever the
//                           atomics did) and gathered: ps = (x,y,z,R_star), vs = (vx,vy,vz,m)
//   nb_contact_cell_kernel  one thread per element in sorted order: own star's grid, then the other's
//                           (skipped when the element is out of reach of that star's bounding box);
//                           fp32 pre-test, survivors queued per lane and evaluated in fp64 in the order found
//
// No library code: the sort is a counting sort by bucket written out here.
#pragma once
#include "nb_kernels.cuh"

namespace nb {

constexpr int kCellScanChunk = 4096;   // counters per block of the prefix sum (1,024 threads x 4)
constexpr int kCellMinDim = 4;         // >= 3, so that the cells of a query are distinct buckets
constexpr float kCellMaxCoord = 1073741824.f;   // 2^30: cell coordinates are clamped to +-this

struct CellGrid {
    float org[3];          // origin of the cell coordinates: the star's mean position
    float inv_h;           // 1 / cell edge (0: no element, or no reach)
    int mx, my, mz;        // table dimensions - 1 (powers of two)
    int sy, sz;            // log2(dim x), log2(dim x * dim y)
    int base;              // first bucket of this star in the table
    int count;             // elements of this star
    float blo[3], bhi[3];  // bounding box of its elements
};

struct CellState { CellGrid g[2]; };

__device__ __forceinline__ int cell_coord(float x, float org, float inv_h) {
    return __float2int_rd(fminf(fmaxf((x - org) * inv_h, -kCellMaxCoord), kCellMaxCoord));
}
__device__ __forceinline__ int cell_bucket(const CellGrid& g, int ix, int iy, int iz) {
    return g.base + (ix & g.mx) + ((iy & g.my) << g.sy) + ((iz & g.mz) << g.sz);
}

// Block b's grid-stride share of star s: part[2 b + s].
struct CellPartial { float lo[3]; int cnt; float hi[3]; float pad0; float sum[3]; float pad1; };

__global__ void __launch_bounds__(256)
nb_cell_bbox_kernel(const float4* __restrict__ posm, int n, int n1, CellPartial* __restrict__ part,
                    int* __restrict__ counters, int ncounters)
{
    __shared__ float sh[2][9][8];
    __shared__ int shc[2][8];
    const int gt = blockIdx.x * blockDim.x + threadIdx.x, stride = gridDim.x * blockDim.x;
    for (int c = gt; c < ncounters; c += stride) counters[c] = 0;
    float q[2][9];
    int cnt[2] = {0, 0};
#pragma unroll
    for (int s = 0; s < 2; ++s)
#pragma unroll
        for (int c = 0; c < 3; ++c) { q[s][c] = 3.0e38f; q[s][3 + c] = -3.0e38f; q[s][6 + c] = 0.f; }
    for (int i = gt; i < n; i += stride) {
        const float4 p = posm[i];
        const float x[3] = {p.x, p.y, p.z};
        const bool first = i < n1;
#pragma unroll
        for (int s = 0; s < 2; ++s) {
            if ((s == 0) == first) {
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    q[s][c] = fminf(q[s][c], x[c]); q[s][3 + c] = fmaxf(q[s][3 + c], x[c]); q[s][6 + c] += x[c];
                }
                ++cnt[s];
            }
        }
    }
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
#pragma unroll
    for (int s = 0; s < 2; ++s) {
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const float a = warp_min(q[s][c]), b = warp_max(q[s][3 + c]);
            float t = q[s][6 + c];
            for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
            if (l == 0) { sh[s][c][w] = a; sh[s][3 + c][w] = b; sh[s][6 + c][w] = t; }
        }
        int k = cnt[s];
        for (int o = 16; o > 0; o >>= 1) k += __shfl_xor_sync(0xffffffffu, k, o);
        if (l == 0) shc[s][w] = k;
    }
    __syncthreads();
    if (threadIdx.x < 2) {
        const int s = threadIdx.x;
        CellPartial r;
        for (int c = 0; c < 3; ++c) {
            float a = sh[s][c][0], b = sh[s][3 + c][0], t = sh[s][6 + c][0];
            for (int k = 1; k < 8; ++k) { a = fminf(a, sh[s][c][k]); b = fmaxf(b, sh[s][3 + c][k]); t += sh[s][6 + c][k]; }
            r.lo[c] = a; r.hi[c] = b; r.sum[c] = t;
        }
        int k = 0;
        for (int j = 0; j < 8; ++j) k += shc[s][j];
        r.cnt = k; r.pad0 = r.pad1 = 0.f;
        part[2 * blockIdx.x + s] = r;
    }
}

// Geometry of star s's grid from the kBoxBlocks partials.  Called by one full warp; the result is the same
// in every lane (xor butterflies) and in every block (same inputs, same order).
__device__ __forceinline__ CellGrid cell_make_grid(const CellPartial* __restrict__ part, int s, float R0, float R1,
                                                   int base, int cap)
{
    const int l = threadIdx.x & 31;
    float lo[3] = {3.0e38f, 3.0e38f, 3.0e38f}, hi[3] = {-3.0e38f, -3.0e38f, -3.0e38f}, sum[3] = {0.f, 0.f, 0.f};
    int cnt = 0;
    for (int b = l; b < kBoxBlocks; b += 32) {
        const CellPartial q = part[2 * b + s];
#pragma unroll
        for (int c = 0; c < 3; ++c) { lo[c] = fminf(lo[c], q.lo[c]); hi[c] = fmaxf(hi[c], q.hi[c]); sum[c] += q.sum[c]; }
        cnt += q.cnt;
    }
    for (int o = 16; o > 0; o >>= 1) cnt += __shfl_xor_sync(0xffffffffu, cnt, o);
    CellGrid g;
    const float h = fmaxf(2.f * (s ? R1 : R0), R0 + R1) * (1.f + 1.0e-5f);
    g.inv_h = (h > 0.f && cnt > 0) ? 1.f / h : 0.f;
    float need[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        lo[c] = warp_min(lo[c]); hi[c] = warp_max(hi[c]);
        float t = sum[c];
        for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
        g.org[c] = cnt > 0 ? t / (float)cnt : 0.f;
        g.blo[c] = lo[c]; g.bhi[c] = hi[c];
        need[c] = cnt > 0 ? fminf((hi[c] - lo[c]) * g.inv_h + 2.f, 1.0e6f) : 1.f;
        if (!(need[c] >= 1.f)) need[c] = 1.f;                    // NaN positions: any grid will do
    }
    int m[3] = {kCellMinDim, kCellMinDim, kCellMinDim};
#pragma unroll
    for (int c = 0; c < 3; ++c) while ((float)m[c] < need[c]) m[c] <<= 1;
    while ((long long)m[0] * m[1] * m[2] > (long long)cap) {     // too many buckets: wrap the longest axis
        int c = 0;
        if (m[1] > m[c]) c = 1;
        if (m[2] > m[c]) c = 2;
        m[c] >>= 1;
    }
    g.mx = m[0] - 1; g.my = m[1] - 1; g.mz = m[2] - 1;
    g.sy = 31 - __clz(m[0]); g.sz = g.sy + 31 - __clz(m[1]);
    g.base = base; g.count = cnt;
    return g;
}

struct CellArgs {
    const float4* __restrict__ posm;
    const float4* __restrict__ vel;
    const DevState* __restrict__ dev;
    const CellPartial* __restrict__ part;
    CellState* __restrict__ cs;        // written by block 0 of nb_cell_count_kernel
    int* __restrict__ counters;        // [ncells + 1]: counts, then first sorted positions
    int* __restrict__ bsum;            // [blocks of the prefix sum]
    int* __restrict__ bucket;          // [n] bucket of element i
    int* __restrict__ slot;            // [n] its arrival number there
    int* __restrict__ tmp;             // [n] element indices by bucket, arrival order
    uint32_t* __restrict__ perm;       // [n] element indices by bucket, index order
    float4* __restrict__ ps;           // [n] x,y,z,R_star   (sorted)
    float4* __restrict__ vs;           // [n] vx,vy,vz,m     (sorted)
    int n, n1, cap0, cap1, ncells;     // cap_s: buckets of star s (a power of two >= 64); ncells = cap0 + cap1
};

__global__ void __launch_bounds__(256)
nb_cell_count_kernel(const __grid_constant__ CellArgs a)
{
    __shared__ CellGrid sg[2];
    const int w = threadIdx.x >> 5;
    if (w < 2) {
        const float R0 = a.dev->R[0], R1 = a.dev->R[1];
        const CellGrid g = cell_make_grid(a.part, w, R0, R1, w ? a.cap0 : 0, w ? a.cap1 : a.cap0);
        if ((threadIdx.x & 31) == 0) {
            sg[w] = g;
            if (blockIdx.x == 0) a.cs->g[w] = g;
        }
    }
    __syncthreads();
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= a.n) return;
    const float4 p = a.posm[i];
    const CellGrid& g = sg[i < a.n1 ? 0 : 1];
    const int b = cell_bucket(g, cell_coord(p.x, g.org[0], g.inv_h), cell_coord(p.y, g.org[1], g.inv_h),
                              cell_coord(p.z, g.org[2], g.inv_h));
    a.bucket[i] = b;
    a.slot[i] = atomicAdd(&a.counters[b], 1);
}

// Exclusive prefix sum of counters[0..ncells) in place, counters[ncells] = total, in two launches of
// ceil(ncells / kCellScanChunk) blocks: phase 0 writes the sum of every chunk; phase 1 adds up the chunk
// sums before its own chunk and scans it.
__global__ void __launch_bounds__(1024)
nb_cell_scan_kernel(int* __restrict__ counters, int* __restrict__ bsum, int ncells, int phase)
{
    __shared__ int wsum[32];
    __shared__ int osum[32];
    const int tid = threadIdx.x, w = tid >> 5, l = tid & 31;
    const int c0 = blockIdx.x * kCellScanChunk + tid * 4;
    int v[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) v[k] = (c0 + k < ncells) ? counters[c0 + k] : 0;
    int inc = v[0] + v[1] + v[2] + v[3];                      // inclusive scan over the threads of the warp
    for (int o = 1; o < 32; o <<= 1) { const int t = __shfl_up_sync(0xffffffffu, inc, o); if (l >= o) inc += t; }
    if (l == 31) wsum[w] = inc;
    int off = 0;                                              // phase 1: chunk sums before this block
    if (phase == 1) {
        for (int b = tid; b < (int)blockIdx.x; b += 1024) off += bsum[b];
        for (int o = 16; o > 0; o >>= 1) off += __shfl_xor_sync(0xffffffffu, off, o);
        if (l == 0) osum[w] = off;
    }
    __syncthreads();
    if (w == 0) {
        int t = wsum[l];                                      // inclusive scan over the warps
        for (int o = 1; o < 32; o <<= 1) { const int u = __shfl_up_sync(0xffffffffu, t, o); if (l >= o) t += u; }
        wsum[l] = t;
        if (phase == 1) {
            int u = osum[l];
            for (int o = 16; o > 0; o >>= 1) u += __shfl_xor_sync(0xffffffffu, u, o);
            osum[l] = u;
        }
    }
    __syncthreads();
    if (phase == 0) {
        if (tid == 0) bsum[blockIdx.x] = wsum[31];
        return;
    }
    int e = osum[0] + (w ? wsum[w - 1] : 0) + inc - (v[0] + v[1] + v[2] + v[3]);   // exclusive prefix of v[0]
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        if (c0 + k < ncells) counters[c0 + k] = e;
        e += v[k];
    }
    if (c0 <= ncells - 1 && ncells - 1 < c0 + 4) counters[ncells] = e;             // the thread owning the last counter
}

__global__ void __launch_bounds__(256)
nb_cell_scatter_kernel(const __grid_constant__ CellArgs a)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < a.n) a.tmp[a.counters[a.bucket[i]] + a.slot[i]] = i;
}

// Sorted position p holds, in arrival order, some element of bucket b; its final place is the number of
// elements of b with a smaller index.  Buckets hold ~1 element (all of a star only when the whole star
// fits into one cell, and then every pair is a candidate anyway).
__global__ void __launch_bounds__(256)
nb_cell_rank_kernel(const __grid_constant__ CellArgs a)
{
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= a.n) return;
    const int idx = a.tmp[p];
    const int b = a.bucket[idx];
    const int s0 = a.counters[b], s1 = a.counters[b + 1];
    int rank = 0;
    for (int q = s0; q < s1; ++q) rank += (a.tmp[q] < idx);
    const int dst = s0 + rank;
    const float4 x = a.posm[idx], v = a.vel[idx];
    a.perm[dst] = (uint32_t)idx;
    a.ps[dst] = make_float4(x.x, x.y, x.z, star_radius(idx, a.n1, a.dev->R[0], a.dev->R[1]));
    a.vs[dst] = make_float4(v.x, v.y, v.z, x.w);
}

struct CellContactArgs {
    const float4* __restrict__ ps;     // [n] x,y,z,R_star   (sorted by star, bucket, index)
    const float4* __restrict__ vs;     // [n] vx,vy,vz,m
    const uint32_t* __restrict__ perm; // [n] original index of sorted element k
    const int* __restrict__ start;     // [ncells + 1] first sorted position of every bucket
    const CellState* __restrict__ cs;
    const DevState* __restrict__ dev;
    float4* __restrict__ out;          // [n] contact acceleration, ORIGINAL index order
    ContactArgs law;                   // gamma, gamma_beta, v_dead, lens_mode (and ps/vs for contact_term's callers)
    int n;
};

constexpr int kCellHitCap = 12;        // per-lane queue of pairs that passed the fp32 pre-test

__global__ void __launch_bounds__(kThreads)
nb_contact_cell_kernel(const __grid_constant__ CellContactArgs a)
{
    __shared__ uint32_t hit_s[kCellHitCap][kThreads];
    const int k = blockIdx.x * kThreads + threadIdx.x;
    if (k >= a.n) return;
    const float4 pi = a.ps[k], vi = a.vs[k];
    const int n0 = a.cs->g[0].count;
    const int si = k < n0 ? 0 : 1;
    const float kSlack = 1.0f + 1.0e-5f;           // the fp32 test is a pre-filter; contact_term() decides in fp64
    double ax = 0.0, ay = 0.0, az = 0.0;
    int nh = 0;
    auto drain = [&]() {
        for (int q = 0; q < nh; ++q) {
            const int j = (int)hit_s[q][threadIdx.x];
            contact_term(a.law, pi, vi, a.ps[j], a.vs[j], ax, ay, az);
        }
        nh = 0;
    };
#pragma unroll 1
    for (int pass = 0; pass < 2; ++pass) {
        const int t = pass ? 1 - si : si;           // own star's grid first, then the other's: a fixed order
        const CellGrid& g = a.cs->g[t];
        if (g.count == 0 || !(g.inv_h > 0.f)) continue;
        const float Rt = a.dev->R[t];
        const float D = (pi.w + Rt) * (1.0f + 1.0e-6f);          // >= R_i + R_j exactly
        if (!(D > 0.f)) continue;
        if (pass) {                                 // out of reach of the other star's bounding box: nothing there
            const float gx = fmaxf(0.f, fmaxf(g.blo[0] - pi.x, pi.x - g.bhi[0]));
            const float gy = fmaxf(0.f, fmaxf(g.blo[1] - pi.y, pi.y - g.bhi[1]));
            const float gz = fmaxf(0.f, fmaxf(g.blo[2] - pi.z, pi.z - g.bhi[2]));
            if (gx * gx + gy * gy + gz * gz > D * D * kSlack) continue;
        }
        const float thr = (pi.w + Rt) * (pi.w + Rt) * kSlack;
        const int x0 = cell_coord(pi.x - D, g.org[0], g.inv_h), x1 = cell_coord(pi.x + D, g.org[0], g.inv_h);
        const int y0 = cell_coord(pi.y - D, g.org[1], g.inv_h), y1 = cell_coord(pi.y + D, g.org[1], g.inv_h);
        const int z0 = cell_coord(pi.z - D, g.org[2], g.inv_h), z1 = cell_coord(pi.z + D, g.org[2], g.inv_h);
        const int nx = min(x1 - x0, g.mx) + 1, ny = min(y1 - y0, g.my) + 1, nz = min(z1 - z0, g.mz) + 1;
#pragma unroll 1
        for (int rz = 0; rz < nz; ++rz) {
#pragma unroll 1
            for (int ry = 0; ry < ny; ++ry) {
                const int row = g.base + (((y0 + ry) & g.my) << g.sy) + (((z0 + rz) & g.mz) << g.sz);
                int c = x0 & g.mx, left = nx;
                while (left > 0) {                  // one range of sorted positions per unwrapped run of cells
                    const int run = min(left, g.mx + 1 - c);
                    const int j0 = a.start[row + c], j1 = a.start[row + c + run];
                    for (int j = j0; j < j1; ++j) {
                        const float4 pj = a.ps[j];
                        const float dx = pj.x - pi.x, dy = pj.y - pi.y, dz = pj.z - pi.z;
                        const float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
                        if (r2 <= thr && j != k) {
                            hit_s[nh][threadIdx.x] = (uint32_t)j;
                            if (++nh == kCellHitCap) drain();
                        }
                    }
                    left -= run; c = 0;
                }
            }
        }
    }
    drain();
    a.out[a.perm[k]] = make_float4((float)ax, (float)ay, (float)az, 0.f);
}

}  // namespace nb
